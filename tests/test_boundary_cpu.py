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


def test_options_and_output_reject_bad_arguments_without_a_device():
    """hsp_set_option / hsp_get_option on the process defaults need no GPU; the library reads no environment."""
    import os
    hsp.reset_options()
    assert hsp.get_option("chol_sb") == -1
    hsp.set_option("chol_sb", 3)
    assert hsp.get_option("chol_sb") == 3
    hsp.set_option("chol_sb", -7)                      # any negative value: automatic
    assert hsp.get_option("chol_sb") == -1
    L = hsp.lib()
    assert L.hsp_set_option(None, b"not_an_option", 1) == -1 and b"unknown option" in L.hsp_last_error()
    v = C.c_longlong()
    assert L.hsp_get_option(None, None, C.byref(v)) == -1
    assert L.hsp_set_output(None, None, None, None, 4) == -1
    assert L.hsp_output_wait(None, None) == -1 and L.hsp_output_ready(None, None) == -1
    hsp.set_option("gram_tc", 1)
    hsp.reset_options()
    assert hsp.get_option("gram_tc") == -1
    src = "".join(open(os.path.join(os.path.dirname(hsp.lib_path()), "csrc", f)).read()
                  for f in os.listdir(os.path.join(os.path.dirname(hsp.lib_path()), "csrc")))
    assert "getenv" not in src


def test_binding_is_marshalling_only():
    """The Python package must not contain the method's arithmetic nor reach for the oracle."""
    import inspect
    import paper_1608_04329_b200.binding as b
    src = inspect.getsource(b)
    assert "oracle" not in src and "erfc" not in src and "cholesky" not in src.lower()
