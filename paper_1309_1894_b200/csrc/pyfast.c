/* _spmvfast: CPython entry point for the hot call of the binding (argument marshalling only).
 *
 * A ctypes call costs ~0.8 us of interpreter work per spmv_apply; for a launch-bound matrix (cfg1: 2 us of
 * kernel) that is a third of the step.  This module forwards (handle, alpha, x, beta, y, stream) -- plain
 * integers and floats -- to the same C ABI function, spmv_apply, through METH_FASTCALL (~0.1 us).
 * Nothing is computed here. */
#define PY_SSIZE_T_CLEAN
#include <Python.h>
#include <stdint.h>

#include "../../include/spmv_b200.h"

static PyObject* fast_apply(PyObject* self, PyObject* const* args, Py_ssize_t nargs) {
  (void)self;
  if (nargs != 6) {
    PyErr_SetString(PyExc_TypeError, "apply(handle, alpha, x_ptr, beta, y_ptr, stream)");
    return NULL;
  }
  void* h = PyLong_AsVoidPtr(args[0]);
  const double alpha = PyFloat_AsDouble(args[1]);
  void* x = PyLong_AsVoidPtr(args[2]);
  const double beta = PyFloat_AsDouble(args[3]);
  void* y = PyLong_AsVoidPtr(args[4]);
  void* stream = PyLong_AsVoidPtr(args[5]);
  if (PyErr_Occurred()) return NULL;
  const spmv_status_t st = spmv_apply((spmv_handle_t)h, alpha, (const double*)x, beta, (double*)y, stream);
  return PyLong_FromLong((long)st);
}

static PyMethodDef methods[] = {
    {"apply", (PyCFunction)(void (*)(void))fast_apply, METH_FASTCALL, "spmv_apply(handle, alpha, x, beta, y, stream) -> status"},
    {NULL, NULL, 0, NULL}};

static struct PyModuleDef module = {PyModuleDef_HEAD_INIT, "_spmvfast", "fast marshalling for spmv_apply", -1, methods,
                                    NULL, NULL, NULL, NULL};

PyMODINIT_FUNC PyInit__spmvfast(void) { return PyModule_Create(&module); }
