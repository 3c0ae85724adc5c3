"""CPU-side checks of the boundary: libhsp.so loads, exports every symbol include/hsp.h declares,
and rejects bad arguments without touching a GPU (no compute calls here)."""
import ctypes as C

import paper_1608_04329_b200 as hsp


def test_library_exports_every_declared_symbol():
    L = hsp.lib()
    names = hsp.declared_symbols()
    assert {"hsp_create", "hsp_sweep", "hsp_get_draws", "hsp_destroy"} <= set(names)
    assert len(names) >= 20
    for n in names:
        assert getattr(L, n) is not None, n


def test_create_rejects_bad_arguments_before_any_device_work():
    L = hsp.lib()
    h = C.c_void_p(123)
    buf = (C.c_double * 8)()
    yb = (C.c_ubyte * 8)()
    assert L.hsp_create(C.byref(h), None, hsp.HSP_F64, yb, 4, 2, 1, None) == -1 and not h.value
    assert b"NULL" in L.hsp_last_error()
    assert L.hsp_create(C.byref(h), buf, 7, yb, 4, 2, 1, None) == -1
    assert L.hsp_create(C.byref(h), buf, hsp.HSP_F64, yb, 1, 2, 1, None) == -1      # N >= 2
    assert L.hsp_create(C.byref(h), buf, hsp.HSP_F64, yb, 4, 0, 1, None) == -1
    # host pointers are not accepted by hsp_create (device pointers only)
    assert L.hsp_create(C.byref(h), buf, hsp.HSP_F64, yb, 4, 2, 1, None) == -1
    assert L.hsp_create(None, buf, hsp.HSP_F64, yb, 4, 2, 1, None) == -1
    assert L.hsp_sweep(None, 1) == -1 and L.hsp_get_draws(None, None, None, None) == -1
    assert L.hsp_destroy(None) == 0


def test_binding_is_marshalling_only():
    """The Python package must not contain the method's arithmetic nor reach for the oracle."""
    import inspect
    import paper_1608_04329_b200.binding as b
    src = inspect.getsource(b)
    assert "oracle" not in src and "erfc" not in src and "cholesky" not in src.lower()
