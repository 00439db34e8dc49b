"""CPU-side checks of the C-ABI library (no GPU): it loads, exports every symbol include/*.h
declare, and its host-only helpers (margins, Eq. 4.2) agree with the oracle's independent versions."""
import ctypes as C
import os
import re

import pytest

import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def ltdi():
    import paper_2505_09600_b200 as m
    m.lib()
    return m


def test_library_exports_every_declared_symbol(ltdi):
    declared = set()
    for name in sorted(os.listdir(os.path.join(ROOT, "include"))):      # lisatdi.h (product) and lisatdi_bench.h (instruments)
        if name.endswith(".h"):
            declared |= set(re.findall(r"\b(ltdi_[a-z0-9_]+)\s*\(", open(os.path.join(ROOT, "include", name)).read()))
    assert declared, "no declarations found"
    handle = C.CDLL(ltdi._build.LIB)
    for name in sorted(declared):
        assert hasattr(handle, name), name
    assert declared == set(ltdi.EXPORTS)


def test_margins_match_the_oracle(ltdi, orc80):
    for dt in (1.0, 5.0, 10.0, 15.0):
        for order in (1, 9, 31, 63):
            for gen in (15, 20):
                for fd in (0, 2, 4):
                    d = W.orbit_desc(100000, dt)
                    assert ltdi.margins(d, gen, order, fd) == orc80.margins(d, gen, order, fd)
                    assert ltdi.link_margins(d, order, fd) == orc80.link_margins(d, order, fd)


def test_hyb_time_matches_the_oracle(ltdi, orc80):
    for M, q, f in ((1e6, 1.0, 2e-3), (1e5, 9.0, 2e-3), (7e6, 3.0, 3e-4)):
        mc = W.chirp_mass_s(M, q)
        a, b = ltdi.hyb_time(f, mc, 2.5e6), orc80.hyb_time(f, mc, 2.5e6)
        assert abs(a - b) <= 1e-9 * abs(2.5e6 - b)


def test_invalid_arguments_are_reported_not_raised_across_the_abi(ltdi):
    lib = ltdi.lib()
    d = ltdi._desc(W.orbit_desc(1000, 5.0))
    lo, hi = C.c_int64(), C.c_int64()
    assert lib.ltdi_margins(C.byref(d), 17, 31, 0, C.byref(lo), C.byref(hi)) == ltdi.EINVAL      # bad generation
    assert lib.ltdi_margins(C.byref(d), 20, 30, 0, C.byref(lo), C.byref(hi)) == ltdi.EINVAL      # even order
    assert lib.ltdi_margins(C.byref(d), 20, 65, 0, C.byref(lo), C.byref(hi)) == ltdi.EINVAL      # order > 63
    assert lib.ltdi_margins(C.byref(d), 20, 31, 3, C.byref(lo), C.byref(hi)) == ltdi.EINVAL      # bad stencil
    nbytes = C.c_size_t()
    bad = ltdi._desc(W.orbit_desc(0, 5.0))
    assert lib.ltdi_orbits_workspace_bytes(C.byref(bad), C.byref(nbytes)) == ltdi.EINVAL
    assert lib.ltdi_orbits_workspace_bytes(C.byref(d), C.byref(nbytes)) == ltdi.OK
    assert nbytes.value == 1024 * (24 * 8 + 16 * 4)     # rows padded to 32: 24 double rows + 16 float rows (low parts)
    out = C.c_double()
    assert lib.ltdi_hyb_time(-1.0, 1.0, 0.0, C.byref(out)) == ltdi.EINVAL
    # NULL required pointers: rejected before any CUDA call
    assert lib.ltdi_response_full(None, None, None, 10, 1, None, 20, 31, None, None, None, None, None, None, 0,
                                  None) == ltdi.EINVAL
    assert lib.ltdi_fp64_probe(None, 1, 1, None, None) == ltdi.EINVAL
    assert ltdi.launch_count() == 0


def test_no_cpu_fallback(ltdi):
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(RuntimeError):
        ltdi.Orbits(W.orbit_desc(100, 5.0))


def test_margins_of_the_next_rows_match_the_oracle(ltdi, orc80):
    """ltdi_margins_lfa_ext (8f-2, third-derivative stencil of the strain) and ltdi_margins_lfa6 ((B30): of the links)"""
    for dt in (5.0, 10.0):
        d = W.orbit_desc(50000, dt)
        for order in (9, 31):
            for gen in (15, 20):
                for fd in (2, 4):
                    for terms in (1, 2):
                        assert ltdi.margins_lfa_ext(d, gen, order, fd, terms) == orc80.margins_lfa_ext(d, gen, order, fd, terms)
                    assert ltdi.margins_lfa6(d, gen, order, fd) == orc80.margins_lfa6(d, gen, order, fd)


def test_next_row_arguments_are_checked_before_any_cuda_call(ltdi):
    lib = ltdi.lib()
    d = ltdi._desc(W.orbit_desc(1000, 5.0))
    lo, hi = C.c_int64(), C.c_int64()
    assert lib.ltdi_margins_lfa_ext(C.byref(d), 20, 31, 2, 3, C.byref(lo), C.byref(hi)) == ltdi.EINVAL     # terms > 2
    assert lib.ltdi_margins_lfa6(C.byref(d), 20, 31, 3, C.byref(lo), C.byref(hi)) == ltdi.EINVAL           # bad stencil
    # numerical orbit file: wrong mode, even knot order, knots that do not cover the grid
    handle = C.c_void_p()
    one = C.c_double(0.0)
    ptr = C.cast(C.byref(one), C.c_void_p)
    kd = ltdi._desc(dict(W.orbit_desc(1000, 5.0), mode=ltdi.ORBIT_KNOTS))
    assert lib.ltdi_orbits_init_knots(C.byref(d), ptr, 40, 0.0, 86400.0, 7, ptr, 1 << 30, None, C.byref(handle)) == ltdi.EINVAL
    assert lib.ltdi_orbits_init_knots(C.byref(kd), ptr, 40, -4 * 86400.0, 86400.0, 6, ptr, 1 << 30, None, C.byref(handle)) == ltdi.EINVAL
    assert lib.ltdi_orbits_init_knots(C.byref(kd), ptr, 40, 86400.0, 86400.0, 7, ptr, 1 << 30, None, C.byref(handle)) == ltdi.EINVAL
    assert lib.ltdi_orbits_init_knots(C.byref(kd), ptr, 6, -4 * 86400.0, 86400.0, 7, ptr, 1 << 30, None, C.byref(handle)) == ltdi.EINVAL
    # waveform model and overlap plan
    assert lib.ltdi_waveform_chirp(None, 1, 0.0, 5.0, 10, 10, None, None, None, 0, None) == ltdi.EINVAL
    assert lib.ltdi_response_full_sagnac(None, ptr, ptr, 10, 1, None, 20, 31, ptr, ptr, ptr, None, None, ptr, 1 << 20, None) == ltdi.EINVAL
    par6 = (C.c_double * 6)(50.0, 0.2, 1e25, 0.3, 0.1, 0.2)
    p6 = C.cast(par6, C.c_void_p)
    assert lib.ltdi_waveform_ecc(ptr, 1, p6, 8, 1, 0.0, 5.0, 10, 10, ptr, ptr, ptr, 64, None) == ltdi.EINVAL      # one knot
    assert lib.ltdi_waveform_ecc(ptr, 16, p6, 65, 1, 0.0, 5.0, 10, 10, ptr, ptr, ptr, 64, None) == ltdi.EINVAL    # > 64 harmonics
    assert lib.ltdi_waveform_ecc(ptr, 16, p6, 8, 1, 0.0, 5.0, 10, 9, ptr, ptr, ptr, 64, None) == ltdi.EINVAL      # ld < n
    assert lib.ltdi_waveform_ecc(ptr, 16, p6, 8, 1, 0.0, 5.0, 10, 10, ptr, ptr, ptr, 63, None) == ltdi.EWORKSPACE
    plan, nbytes = C.c_void_p(), C.c_size_t()
    assert lib.ltdi_overlap_create(1, 1, 1, C.byref(plan), C.byref(nbytes)) == ltdi.EINVAL                # n < 2
    assert lib.ltdi_overlap_create(40007, 40007, 3, C.byref(plan), C.byref(nbytes)) == ltdi.OK            # a prime: Bluestein, m = 2^17
    assert nbytes.value >= (40007 + 2 * 131072 + 2 * 9 * 131072) * 16
    assert lib.ltdi_overlap_destroy(plan) == ltdi.OK
    assert lib.ltdi_overlap_create(131072, 131072, 2, C.byref(plan), C.byref(nbytes)) == ltdi.OK          # a power of two: no chirp tables
    assert nbytes.value < (2 * 6 * 131072 + 4096) * 16 + (1 << 16)
    assert lib.ltdi_overlap_destroy(plan) == ltdi.OK
    assert ltdi.launch_count() == 0
