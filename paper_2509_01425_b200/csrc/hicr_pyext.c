/* hicr_pyext.c -- CPython entry points for the calls of a step (argument marshalling only).
 *
 * binding.py marshals every call of include/hicr.h with ctypes; that costs about a
 * microsecond per call on the host, which is on the critical path of a step that ends in a
 * blocking fence (config 1: 14 us per step; config 5a through push/pop: 65 k calls).  The
 * calls a step consists of -- hicr_memcpy_batch, hicr_fence, hicr_fence_async,
 * hicr_channel_push, hicr_channel_pop -- are therefore also exported here through the
 * CPython C API (METH_FASTCALL, ~0.1 us per call).  Handles and addresses are plain ints.
 * Nothing but marshalling happens in this file: every function forwards to the C ABI of
 * libhicr_b200.so and returns its status.
 */
#define PY_SSIZE_T_CLEAN
#include <Python.h>
#include <stdint.h>

#include "hicr.h"

static int as_u64(PyObject *o, uint64_t *out)
{
    const unsigned long long v = PyLong_AsUnsignedLongLong(o);
    if (v == (unsigned long long)-1 && PyErr_Occurred()) return 0;
    *out = (uint64_t)v;
    return 1;
}

static int want(Py_ssize_t nargs, Py_ssize_t n, const char *name)
{
    if (nargs == n) return 1;
    PyErr_Format(PyExc_TypeError, "%s takes %zd arguments (%zd given)", name, n, nargs);
    return 0;
}

/* memcpy_batch(ctx, descs_address, n, descs_on_device) -> (status, first_bad) on error, 0 on success */
static PyObject *py_memcpy_batch(PyObject *self, PyObject *const *args, Py_ssize_t nargs)
{
    uint64_t h, p, n, dev, bad = 0;
    int rc;
    (void)self;
    if (!want(nargs, 4, "memcpy_batch")) return NULL;
    if (!as_u64(args[0], &h) || !as_u64(args[1], &p) || !as_u64(args[2], &n) || !as_u64(args[3], &dev)) return NULL;
    Py_BEGIN_ALLOW_THREADS
    rc = hicr_memcpy_batch((hicr_ctx_t *)(uintptr_t)h, (const hicr_desc_t *)(uintptr_t)p, n, (int)dev, &bad);
    Py_END_ALLOW_THREADS
    if (rc == HICR_OK) return PyLong_FromLong(0);
    return Py_BuildValue("(iK)", rc, (unsigned long long)bad);
}

/* fence(ctx) -> status */
static PyObject *py_fence(PyObject *self, PyObject *const *args, Py_ssize_t nargs)
{
    uint64_t h;
    int rc;
    (void)self;
    if (!want(nargs, 1, "fence")) return NULL;
    if (!as_u64(args[0], &h)) return NULL;
    Py_BEGIN_ALLOW_THREADS
    rc = hicr_fence((hicr_ctx_t *)(uintptr_t)h);
    Py_END_ALLOW_THREADS
    return PyLong_FromLong(rc);
}

/* fence_async(ctx) -> status */
static PyObject *py_fence_async(PyObject *self, PyObject *const *args, Py_ssize_t nargs)
{
    uint64_t h;
    (void)self;
    if (!want(nargs, 1, "fence_async")) return NULL;
    if (!as_u64(args[0], &h)) return NULL;
    return PyLong_FromLong(hicr_fence_async((hicr_ctx_t *)(uintptr_t)h));
}

/* channel_push(channel, slot, offset, n_tokens) / channel_pop(channel, slot, offset, max_tokens)
 * -> tokens moved (>= 0), or the negative status */
static PyObject *channel_call(PyObject *const *args, Py_ssize_t nargs, int push)
{
    uint64_t h, slot, off, n, k = 0;
    int rc;
    if (!want(nargs, 4, push ? "channel_push" : "channel_pop")) return NULL;
    if (!as_u64(args[0], &h) || !as_u64(args[1], &slot) || !as_u64(args[2], &off) || !as_u64(args[3], &n)) return NULL;
    Py_BEGIN_ALLOW_THREADS
    rc = push ? hicr_channel_push((hicr_channel_t *)(uintptr_t)h, (hicr_slot_t)slot, off, n, &k)
              : hicr_channel_pop((hicr_channel_t *)(uintptr_t)h, (hicr_slot_t)slot, off, n, &k);
    Py_END_ALLOW_THREADS
    if (rc != HICR_OK) return PyLong_FromLong(rc);
    return PyLong_FromUnsignedLongLong((unsigned long long)k);
}
static PyObject *py_channel_push(PyObject *self, PyObject *const *args, Py_ssize_t nargs)
{
    (void)self;
    return channel_call(args, nargs, 1);
}
static PyObject *py_channel_pop(PyObject *self, PyObject *const *args, Py_ssize_t nargs)
{
    (void)self;
    return channel_call(args, nargs, 0);
}

static PyMethodDef methods[] = {
    {"memcpy_batch", (PyCFunction)(void (*)(void))py_memcpy_batch, METH_FASTCALL, "hicr_memcpy_batch"},
    {"fence", (PyCFunction)(void (*)(void))py_fence, METH_FASTCALL, "hicr_fence"},
    {"fence_async", (PyCFunction)(void (*)(void))py_fence_async, METH_FASTCALL, "hicr_fence_async"},
    {"channel_push", (PyCFunction)(void (*)(void))py_channel_push, METH_FASTCALL, "hicr_channel_push"},
    {"channel_pop", (PyCFunction)(void (*)(void))py_channel_pop, METH_FASTCALL, "hicr_channel_pop"},
    {NULL, NULL, 0, NULL},
};

static struct PyModuleDef moduledef = {PyModuleDef_HEAD_INIT, "_hicr_step", "hot calls of include/hicr.h", -1, methods,
                                       NULL, NULL, NULL, NULL};

PyMODINIT_FUNC PyInit__hicr_step(void) { return PyModule_Create(&moduledef); }
