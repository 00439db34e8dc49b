"""paper_2505_09600_b200 -- thin Python binding of liblisatdi.so (include/lisatdi.h).

Argument marshalling only: every step of the response runs in the CUDA kernels of
csrc/.  PyTorch supplies device memory and streams.  There is no CPU fallback: a
missing library or a missing GPU raises.

    import paper_2505_09600_b200 as ltdi
    orb = ltdi.Orbits(ltdi.orbit_desc(n, dt, ltdi.ORBIT_KEPLERIAN))       # orbit/delay kernel
    out = ltdi.response_full(orb, hp, hc, sources, gen=20, order=31)      # dict of device tensors
    out = ltdi.response_lfa(orb, hp, hc, sources, gen=20, order=31, fd_order=2)
    out = ltdi.response_hybrid(orb, hp, hc, sources, 20, 31, 2, hybrid=[{...}])

hp, hc: float64 CUDA tensors [batch][ld]; sources: [batch][3] (beta, lambda, psi), host.
"""
import ctypes as C
import os

import torch

from . import build as _build

GEN_15, GEN_20 = 15, 20
ORBIT_STATIC_EQUALARM, ORBIT_KEPLERIAN, ORBIT_TABLES, ORBIT_KNOTS = 0, 1, 2, 3
TAPER_SIGMOID, TAPER_COSINE = 0, 1
RESPONSE_FULL, RESPONSE_LFA, RESPONSE_HYBRID = 0, 1, 2
LFA_CENTRAL, LFA_BACKWARD, LFA_FORWARD = 0, 1, 2
OK, EINVAL, EUNSUPPORTED, ECUDA, EWORKSPACE = 0, -1, -2, -3, -4
_ERR = {EINVAL: "LTDI_EINVAL", EUNSUPPORTED: "LTDI_EUNSUPPORTED", ECUDA: "LTDI_ECUDA",
        EWORKSPACE: "LTDI_EWORKSPACE"}

C_LIGHT = 299792458.0
ARM_M = 2.5e9
AU_M = 149597870700.0
YEAR_S = 31558149.7635      # sidereal year; Omega = 2 pi / yr


class LtdiError(RuntimeError):
    def __init__(self, fn, code):
        super().__init__(f"{fn}: {_ERR.get(code, code)}")
        self.code = code


class OrbitDesc(C.Structure):
    _fields_ = [("t0", C.c_double), ("dt", C.c_double), ("n", C.c_int64), ("arm_m", C.c_double),
                ("R_m", C.c_double), ("period_s", C.c_double), ("alpha0", C.c_double),
                ("rot0", C.c_double), ("mode", C.c_int32)]


class Source(C.Structure):
    _fields_ = [("beta", C.c_double), ("lam", C.c_double), ("psi", C.c_double)]


class Chirp(C.Structure):
    _fields_ = [("t_c", C.c_double), ("mc_s", C.c_double), ("dist_m", C.c_double), ("cos_iota", C.c_double),
                ("phi_c", C.c_double), ("tau_cut", C.c_double), ("f_rd", C.c_double), ("tau_rd", C.c_double)]


CHIRP_KEYS = ("t_c", "mc_s", "dist_m", "cos_iota", "phi_c", "tau_cut", "f_rd", "tau_rd")


def _chirps(params):
    arr = (Chirp * len(params))()
    for i, p in enumerate(params):
        arr[i] = Chirp(*[float(p[k]) for k in CHIRP_KEYS])
    return arr


class Hybrid(C.Structure):
    _fields_ = [("t_hyb", C.c_double), ("window_s", C.c_double), ("sigma_s", C.c_double),
                ("taper", C.c_int32)]


_vp, _dp, _i64p, _szp = C.c_void_p, C.c_void_p, C.POINTER(C.c_int64), C.POINTER(C.c_size_t)
_SIGNATURES = {
    "ltdi_orbits_workspace_bytes": (C.c_int, [C.POINTER(OrbitDesc), _szp]),
    "ltdi_orbits_init": (C.c_int, [C.POINTER(OrbitDesc), _vp, C.c_size_t, _vp, C.POINTER(_vp)]),
    "ltdi_orbits_init_tables": (C.c_int, [C.POINTER(OrbitDesc), _dp, _dp, _vp, C.c_size_t, _vp, C.POINTER(_vp)]),
    "ltdi_orbits_init_knots": (C.c_int, [C.POINTER(OrbitDesc), _dp, C.c_int64, C.c_double, C.c_double, C.c_int, _vp,
                                         C.c_size_t, _vp, C.POINTER(_vp)]),
    "ltdi_orbits_prepare_bytes": (C.c_int, [C.POINTER(OrbitDesc), C.c_int, _szp]),
    "ltdi_orbits_prepare": (C.c_int, [_vp, C.c_int, C.c_int, _vp, C.c_size_t, _vp]),
    "ltdi_orbits_destroy": (C.c_int, [_vp]),
    "ltdi_orbits_stride": (C.c_int64, [_vp]),
    "ltdi_orbits_tables": (_vp, [_vp]),
    "ltdi_margins": (C.c_int, [C.POINTER(OrbitDesc), C.c_int, C.c_int, C.c_int, _i64p, _i64p]),
    "ltdi_link_margins": (C.c_int, [C.POINTER(OrbitDesc), C.c_int, C.c_int, _i64p, _i64p]),
    "ltdi_hyb_time": (C.c_int, [C.c_double, C.c_double, C.c_double, C.POINTER(C.c_double)]),
    "ltdi_workspace_bytes": (C.c_int, [C.c_int, C.c_int64, C.c_int64, C.c_int, C.c_int, _szp]),
    "ltdi_response_full": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                     _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_response_static": (C.c_int, [C.c_int, _vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int, C.c_int,
                                       C.POINTER(Hybrid), C.c_int64, _dp, _dp, _dp, _vp]),
    "ltdi_response_full_sagnac": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                            _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_response_full_nested": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int, C.c_int,
                                            _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_waveform_chirp": (C.c_int, [C.POINTER(Chirp), C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_int64, _dp, _dp, _vp,
                                      C.c_size_t, _vp]),
    "ltdi_waveform_ecc": (C.c_int, [_dp, C.c_int64, _dp, C.c_int, C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_int64, _dp, _dp,
                                    _vp, C.c_size_t, _vp]),
    "ltdi_response_full_chirp": (C.c_int, [_vp, C.POINTER(Chirp), C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                           _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_response_lfa": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                    C.c_int, _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_response_lfa_ext": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                        C.c_int, C.c_int, C.c_int, _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_response_lfa6": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int, C.c_int,
                                     _dp, _dp, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_margins_lfa6": (C.c_int, [C.POINTER(OrbitDesc), C.c_int, C.c_int, C.c_int, _i64p, _i64p]),
    "ltdi_margins_lfa_ext": (C.c_int, [C.POINTER(OrbitDesc), C.c_int, C.c_int, C.c_int, C.c_int, _i64p, _i64p]),
    "ltdi_response_hybrid": (C.c_int, [_vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                       C.c_int, C.POINTER(Hybrid), C.c_int64, _dp, _dp, _dp, _dp, _dp, _vp,
                                       C.c_size_t, _vp]),
    "ltdi_host_scratch_bytes": (C.c_int, [C.c_int64, C.c_int64, _szp]),
    "ltdi_response_host": (C.c_int, [C.c_int, _vp, _dp, _dp, C.c_int64, C.c_int64, C.POINTER(Source), C.c_int, C.c_int,
                                     C.c_int, C.POINTER(Hybrid), C.c_int64, _dp, _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_noise_psd": (C.c_int, [C.c_void_p, C.c_double, C.c_int64, _dp, _vp]),
    "ltdi_overlap_create": (C.c_int, [C.c_int64, C.c_int64, C.c_int64, C.POINTER(_vp), _szp]),
    "ltdi_overlap_destroy": (C.c_int, [_vp]),
    "ltdi_overlap_products": (C.c_int, [_vp, _dp, _dp, _dp, _dp, _dp, _dp, C.c_double, _dp, C.c_double, C.c_double,
                                        _dp, _dp, _vp, C.c_size_t, _vp]),
    "ltdi_fp64_probe": (C.c_int, [_dp, C.c_int, C.c_int, _vp, C.POINTER(C.c_double)]),
    "ltdi_profile_enable": (C.c_int, [C.c_int]),
    "ltdi_profile_read": (C.c_int, [C.c_int, C.c_int, C.POINTER(C.c_double), _i64p]),
    "ltdi_profile_reset": (C.c_int, []),
    "ltdi_launch_count": (C.c_int64, []),
    "ltdi_profile_slow_tiles": (C.c_int, [_i64p, C.c_int]),
    "ltdi_version": (C.c_char_p, []),
}
EXPORTS = tuple(_SIGNATURES)

_lib = None


def lib():
    """Load (building first if the sources are newer) liblisatdi.so; raises if that fails."""
    global _lib
    if _lib is None:
        path = os.environ.get("LTDI_LIBRARY") or _build.build()   # LTDI_LIBRARY: an already built liblisatdi.so to load instead
        handle = C.CDLL(path)
        for name, (res, args) in _SIGNATURES.items():
            fn = getattr(handle, name)   # AttributeError if the library does not export it
            fn.restype, fn.argtypes = res, args
        _lib = handle
    return _lib


def _check(fn, code):
    if code != OK:
        raise LtdiError(fn, code)


def orbit_desc(n, dt, mode=ORBIT_KEPLERIAN, t0=0.0, arm_m=ARM_M, R_m=AU_M, period_s=YEAR_S, alpha0=0.0,
               rot0=0.0):
    return {"t0": float(t0), "dt": float(dt), "n": int(n), "arm_m": float(arm_m), "R_m": float(R_m),
            "period_s": float(period_s), "alpha0": float(alpha0), "rot0": float(rot0), "mode": int(mode)}


def _desc(d):
    return OrbitDesc(d["t0"], d["dt"], int(d["n"]), d["arm_m"], d["R_m"], d["period_s"], d["alpha0"], d["rot0"],
                     int(d["mode"]))


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def _dev_f64(t, name):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous float64 CUDA tensor")
    return t


def margins(desc, gen, order, fd_order=0):
    lo, hi = C.c_int64(), C.c_int64()
    d = _desc(desc)
    _check("ltdi_margins", lib().ltdi_margins(C.byref(d), gen, order, fd_order, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def time_shard(desc, lo, hi, world, rank):
    """the piece of ONE long series that rank `rank` of `world` computes -- the path needs no exchange step, a
    piece only re-reads a halo of the input.  The valid outputs [lo, n - hi) (lo, hi from margins() of the response at
    hand) are split into `world` contiguous runs [a, b); the rank evaluates the response on the sub-grid that starts lo
    samples before a and ends hi samples after b, whose own valid range is exactly [a, b).
    Returns (sub_desc, src, dst, a, b): sub_desc = desc with t0 and n of the sub-grid (tabulated orbits sliced with it; a
    numerical orbit file keeps its knots), src = slice of the input samples the rank reads, dst = slice of the sub-grid's
    output that holds the global samples [a, b).  Pure host logic: no CUDA call."""
    n = int(desc["n"])
    world, rank = int(world), int(rank)
    if world < 1 or not 0 <= rank < world or lo < 0 or hi < 0 or n - hi - lo < world:
        raise ValueError("time_shard: needs 0 <= rank < world <= number of valid samples")
    valid = n - hi - lo
    a = lo + valid * rank // world
    b = lo + valid * (rank + 1) // world
    first, last = a - lo, b + hi                     # input samples [first, last)
    sub = dict(desc, t0=float(desc["t0"]) + first * float(desc["dt"]), n=last - first)
    for key in ("R_table", "L_table"):               # ORBIT_TABLES: per-sample tables travel with the grid
        if key in sub and sub[key] is not None:
            sub[key] = sub[key][..., first:last]
    return sub, slice(first, last), slice(lo, lo + (b - a)), a, b


def margins_lfa_ext(desc, gen, order, fd_order, terms=1):
    lo, hi = C.c_int64(), C.c_int64()
    d = _desc(desc)
    _check("ltdi_margins_lfa_ext", lib().ltdi_margins_lfa_ext(C.byref(d), gen, order, fd_order, terms, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def link_margins(desc, order, fd_order=0):
    lo, hi = C.c_int64(), C.c_int64()
    d = _desc(desc)
    _check("ltdi_link_margins", lib().ltdi_link_margins(C.byref(d), order, fd_order, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def hyb_time(f_hyb_hz, mchirp_s, t_c):
    out = C.c_double()
    _check("ltdi_hyb_time", lib().ltdi_hyb_time(f_hyb_hz, mchirp_s, t_c, C.byref(out)))
    return out.value


def slow_tiles(reset=True):
    """(TDI tile, channel) pairs that fell back to exact per-sample weights since the last reset (diagnostic)."""
    n = C.c_int64()
    _check("ltdi_profile_slow_tiles", lib().ltdi_profile_slow_tiles(C.byref(n), int(bool(reset))))
    return n.value


def launch_count():
    return lib().ltdi_launch_count()


KERNELS = ("orbit", "prep", "anchor", "link_full", "link_lfa", "tdi", "generic", "tdi_lfa", "plan")   # LTDI_KERNEL_* order


def profile_enable(on=True):
    _check("ltdi_profile_enable", lib().ltdi_profile_enable(int(bool(on))))


def profile_reset():
    _check("ltdi_profile_reset", lib().ltdi_profile_reset())


def profile_read():
    """{response: {kernel name: (device ms accumulated, launches)}} from the library's per-kernel CUDA events."""
    out = {}
    for w, resp in enumerate(("full", "lfa", "hybrid")):
        out[resp] = {}
        for i, name in enumerate(KERNELS):
            ms, n = C.c_double(), C.c_int64()
            _check("ltdi_profile_read", lib().ltdi_profile_read(i, w, C.byref(ms), C.byref(n)))
            if n.value:
                out[resp][name] = (ms.value, n.value)
    return out


class Orbits:
    """Device orbit tables for one time grid (S0, the orbit/delay kernel)."""

    def __init__(self, desc, R_table=None, L_table=None, device="cuda:0", knots=None):
        """desc: orbit_desc dict.  ORBIT_TABLES: R_table [3][3][n], L_table [6][n] device tensors.  ORBIT_KNOTS (a numerical
        orbit file): knots [3][3][nk] device tensor (default: desc["knots"] uploaded) with desc["knot_t0"], ["knot_dt"],
        ["knot_order"]."""
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2505_09600_b200 needs a CUDA device (no CPU fallback)")
        self.desc = dict(desc)
        self.device = torch.device(device)
        d = _desc(desc)
        nbytes = C.c_size_t()
        _check("ltdi_orbits_workspace_bytes", lib().ltdi_orbits_workspace_bytes(C.byref(d), C.byref(nbytes)))
        self.tables = torch.empty(nbytes.value // 8, dtype=torch.float64, device=self.device)
        handle = C.c_void_p()
        with torch.cuda.device(self.device):
            if int(desc["mode"]) == ORBIT_KNOTS:
                if knots is None:
                    knots = torch.as_tensor(desc["knots"], dtype=torch.float64).contiguous().to(self.device)
                self._knots = _dev_f64(knots, "knots")
                assert self._knots.dim() == 3 and tuple(self._knots.shape[:2]) == (3, 3)
                rc = lib().ltdi_orbits_init_knots(C.byref(d), self._knots.data_ptr(), int(self._knots.shape[2]),
                                                  float(desc["knot_t0"]), float(desc["knot_dt"]), int(desc["knot_order"]),
                                                  self.tables.data_ptr(), nbytes.value, _stream(), C.byref(handle))
            elif int(desc["mode"]) == ORBIT_TABLES:
                self._R = _dev_f64(R_table, "R_table")   # [3][3][n]
                self._L = _dev_f64(L_table, "L_table")   # [6][n]
                assert self._R.shape == (3, 3, d.n) and self._L.shape == (6, d.n)
                rc = lib().ltdi_orbits_init_tables(C.byref(d), self._R.data_ptr(), self._L.data_ptr(),
                                                   self.tables.data_ptr(), nbytes.value, _stream(), C.byref(handle))
            else:
                rc = lib().ltdi_orbits_init(C.byref(d), self.tables.data_ptr(), nbytes.value, _stream(),
                                            C.byref(handle))
        _check("ltdi_orbits_init", rc)
        self.handle = handle
        self.stride = lib().ltdi_orbits_stride(handle)
        self._anchors = None

    def prepare(self, gen, order, buffer=None):
        """Compute the TDI-stage interpolation weights of (gen, order) once for this time grid
        (ltdi_orbits_prepare); later responses with the same gen and order skip their weight kernel.
        `buffer`: an existing float64 device tensor to reuse (a new one is allocated if None or too small)."""
        nbytes = C.c_size_t()
        _check("ltdi_orbits_prepare_bytes",
               lib().ltdi_orbits_prepare_bytes(C.byref(_desc(self.desc)), order, C.byref(nbytes)))
        if nbytes.value == 0:
            return self
        if buffer is None or buffer.numel() * 8 < nbytes.value:
            buffer = torch.empty(nbytes.value // 8, dtype=torch.float64, device=self.device)
        self._anchors = buffer
        with torch.cuda.device(self.device):
            _check("ltdi_orbits_prepare", lib().ltdi_orbits_prepare(self.handle, gen, order, buffer.data_ptr(),
                                                                   buffer.numel() * 8, _stream()))
        return self

    @property
    def n(self):
        return int(self.desc["n"])

    def rows(self):
        """[24][n] view of the table: R (9 rows), n_l for l = +1,+2,+3 (9 rows), L_l (6 rows)."""
        return self.tables[:24 * self.stride].view(24, self.stride)[:, :self.n]

    def rows_lo(self):
        """[15][n] float32 view: low parts of the double-double n_l (9 rows) and L_l (6 rows) of the table."""
        return self.tables[24 * self.stride:].view(torch.float32).view(16, self.stride)[:15, :self.n]

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:
            _lib.ltdi_orbits_destroy(h)


def _sources(sources):
    s = torch.as_tensor(sources, dtype=torch.float64, device="cpu").reshape(-1, 3).contiguous()
    return C.cast(C.c_void_p(s.data_ptr()), C.POINTER(Source)), s   # same layout as ltdi_source[batch]


class Workspace:
    """Preallocated outputs and scratch so that repeated calls allocate nothing."""

    def __init__(self, batch, ld, device, want_xyz=False, want_y=False):
        kw = dict(dtype=torch.float64, device=device)
        self.A, self.E, self.T = (torch.empty(batch, ld, **kw) for _ in range(3))
        self.XYZ = torch.empty(3, batch, ld, **kw) if want_xyz else None
        self.y = torch.empty(6, batch, ld, **kw) if want_y else None
        need = 0   # one scratch buffer that serves every response (the chunking differs per response)
        for which in (RESPONSE_FULL, RESPONSE_LFA, RESPONSE_HYBRID):
            nbytes = C.c_size_t()
            _check("ltdi_workspace_bytes", lib().ltdi_workspace_bytes(which, ld, batch, GEN_20, 31, C.byref(nbytes)))
            need = max(need, nbytes.value)
        self.work = torch.empty(need // 8, **kw)

    def outputs(self):
        return {"A": self.A, "E": self.E, "T": self.T, "XYZ": self.XYZ, "y": self.y}


def _run(which, orb, hp, hc, sources, gen, order, fd_order, hybrid, want_xyz, want_y, ws, ext=None):
    hp, hc = _dev_f64(hp, "hp"), _dev_f64(hc, "hc")
    if hp.dim() == 1:
        hp, hc = hp[None], hc[None]
    batch, ld = hp.shape
    assert hc.shape == hp.shape
    src_ptr, keep = _sources(sources)
    assert keep.shape[0] == batch, "one (beta, lambda, psi) per source"
    if ws is None:
        ws = Workspace(batch, ld, hp.device, want_xyz, want_y)
    p = lambda t: None if t is None else t.data_ptr()
    head = [orb.handle, hp.data_ptr(), hc.data_ptr(), ld, batch, src_ptr, gen, order]
    with torch.cuda.device(hp.device):
        # the stream handle must be the current stream of the tensors' device: evaluated inside the device context
        tail = [p(ws.A), p(ws.E), p(ws.T), p(ws.XYZ), p(ws.y), ws.work.data_ptr(), ws.work.numel() * 8, _stream()]
        if which == RESPONSE_FULL and ext == "sagnac":
            rc, fn = lib().ltdi_response_full_sagnac(*head, *tail), "ltdi_response_full_sagnac"
        elif which == RESPONSE_FULL and ext is not None:
            rc, fn = lib().ltdi_response_full_nested(*head, int(ext[0]), *tail), "ltdi_response_full_nested"
        elif which == RESPONSE_FULL:
            rc, fn = lib().ltdi_response_full(*head, *tail), "ltdi_response_full"
        elif which == RESPONSE_LFA and ext == "lfa6":
            rc, fn = lib().ltdi_response_lfa6(*head, fd_order, *tail), "ltdi_response_lfa6"
        elif which == RESPONSE_LFA and ext is not None:
            rc, fn = lib().ltdi_response_lfa_ext(*head, fd_order, int(ext[0]), int(ext[1]), *tail), "ltdi_response_lfa_ext"
        elif which == RESPONSE_LFA:
            rc, fn = lib().ltdi_response_lfa(*head, fd_order, *tail), "ltdi_response_lfa"
        else:
            hl = hybrid if isinstance(hybrid, (list, tuple)) else [hybrid]
            harr = (Hybrid * len(hl))(*[Hybrid(h["t_hyb"], h["window_s"], h["sigma_s"], int(h["taper"])) for h in hl])
            rc, fn = lib().ltdi_response_hybrid(*head, fd_order, harr, len(hl), *tail), "ltdi_response_hybrid"
    _check(fn, rc)
    return ws.outputs()


def response_full(orb, hp, hc, sources, gen, order, want_xyz=False, want_y=False, workspace=None):
    """Eqs. (2.2)-(2.9): projection, TDI `gen`, A, E, T.  Returns dict A, E, T (, XYZ, y)."""
    return _run(RESPONSE_FULL, orb, hp, hc, sources, gen, order, 0, None, want_xyz, want_y, workspace)


def response_full_sagnac(orb, hp, hc, sources, gen, order, want_abc=False, want_y=False, workspace=None):
    """the full response in the Sagnac combinations; "XYZ" of the result holds alpha, beta, gamma, and A, E, T
    are Eq. (2.9) applied to them (ltdi_response_full_sagnac)."""
    return _run(RESPONSE_FULL, orb, hp, hc, sources, gen, order, 0, None, want_abc, want_y, workspace, ext="sagnac")


def response_full_nested(orb, hp, hc, sources, gen, order, nested_order=3, want_xyz=False, want_y=False, workspace=None):
    """the full response with properly nested TDI delays (light times looked up by Lagrange order 3)."""
    return _run(RESPONSE_FULL, orb, hp, hc, sources, gen, order, 0, None, want_xyz, want_y, workspace, ext=(nested_order,))


def waveform_chirp(params, t0, dt, n, device="cuda:0", out=None):
    """the chirp + ringdown model of `params` (list of dicts, CHIRP_KEYS) sampled on t0 + i dt on the device:
    returns hp, hc [batch][n] float64 device tensors (ltdi_waveform_chirp)."""
    batch = len(params)
    dev = torch.device(device)
    hp, hc = out if out is not None else (torch.empty(batch, n, dtype=torch.float64, device=dev) for _ in range(2))
    work = torch.empty(batch * 20, dtype=torch.float64, device=dev)
    with torch.cuda.device(dev):
        _check("ltdi_waveform_chirp", lib().ltdi_waveform_chirp(_chirps(params), batch, float(t0), float(dt), int(n), int(hp.shape[1]),
                                                                hp.data_ptr(), hc.data_ptr(), work.data_ptr(), work.numel() * 8, _stream()))
    return hp, hc


def waveform_ecc(tables, params, nharm, t0, dt, n, out=None):
    """the eccentric harmonic-sum model on the device.  tables: float64 CUDA tensor [batch][7][nk] (t, F, e, l and
    their time derivatives at the knots); params: host array [batch][6] (M_s, eta, dist_m, cos_iota, gamma, l0).
    Returns hp, hc [batch][n] device tensors (ltdi_waveform_ecc)."""
    tab = _dev_f64(tables, "tables")
    batch, seven, nk = tab.shape
    assert seven == 7
    par = torch.as_tensor(params, dtype=torch.float64, device="cpu").reshape(batch, 6).contiguous()
    hp, hc = out if out is not None else (torch.empty(batch, n, dtype=torch.float64, device=tab.device) for _ in range(2))
    work = torch.empty(batch * 8, dtype=torch.float64, device=tab.device)
    with torch.cuda.device(tab.device):
        _check("ltdi_waveform_ecc", lib().ltdi_waveform_ecc(tab.data_ptr(), int(nk), par.data_ptr(), int(nharm), batch, float(t0), float(dt),
                                                            int(n), int(hp.shape[1]), hp.data_ptr(), hc.data_ptr(), work.data_ptr(),
                                                            work.numel() * 8, _stream()))
    return hp, hc


def response_full_chirp(orb, params, sources, gen, order, want_xyz=False, want_y=False, workspace=None):
    """full response from waveform parameters, the model evaluated at the retarded times of Eq. (2.5)."""
    batch, ld = len(params), orb.n
    src_ptr, keep = _sources(sources)
    assert keep.shape[0] == batch
    ws = workspace or Workspace(batch, ld, orb.device, want_xyz, want_y)
    p = lambda t: None if t is None else t.data_ptr()
    with torch.cuda.device(orb.device):
        rc = lib().ltdi_response_full_chirp(orb.handle, _chirps(params), ws.A.shape[1], batch, src_ptr, gen, order, p(ws.A), p(ws.E),
                                            p(ws.T), p(ws.XYZ), p(ws.y), ws.work.data_ptr(), ws.work.numel() * 8, _stream())
    _check("ltdi_response_full_chirp", rc)
    return ws.outputs()


def response_lfa(orb, hp, hc, sources, gen, order, fd_order, want_xyz=False, want_y=False, workspace=None):
    """Eqs. (B10), (B25)/(B33): low-frequency approximation with central stencils of order fd_order."""
    return _run(RESPONSE_LFA, orb, hp, hc, sources, gen, order, fd_order, None, want_xyz, want_y, workspace)


def response_lfa_ext(orb, hp, hc, sources, gen, order, fd_order, terms=1, point=LFA_CENTRAL, want_xyz=False,
                     want_y=False, workspace=None):
    """`terms` terms of the single-link series Eq. (B4) about the expansion point `point`
    (LFA_CENTRAL (B1), LFA_BACKWARD (B13), LFA_FORWARD (B14)), then (B25) / (B33)."""
    return _run(RESPONSE_LFA, orb, hp, hc, sources, gen, order, fd_order, None, want_xyz, want_y, workspace,
                ext=(terms, point))


def response_lfa6(orb, hp, hc, sources, gen, order, fd_order, want_xyz=False, want_y=False, workspace=None):
    """six LFA links and the Michelson variables of Eq. (B20) / (B30) (no link-reversal symmetry)."""
    return _run(RESPONSE_LFA, orb, hp, hc, sources, gen, order, fd_order, None, want_xyz, want_y, workspace, ext="lfa6")


def margins_lfa6(desc, gen, order, fd_order):
    lo, hi = C.c_int64(), C.c_int64()
    d = _desc(desc)
    _check("ltdi_margins_lfa6", lib().ltdi_margins_lfa6(C.byref(d), gen, order, fd_order, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def response_hybrid(orb, hp, hc, sources, gen, order, fd_order, hybrid, want_xyz=False, want_y=False,
                    workspace=None):
    """Eqs. (4.5), (4.6): LFA spliced to the full response; hybrid = dict or list of dicts
    {t_hyb, window_s, sigma_s, taper}."""
    return _run(RESPONSE_HYBRID, orb, hp, hc, sources, gen, order, fd_order, hybrid, want_xyz, want_y, workspace)


def _hybrid_array(hybrid):
    if hybrid is None:
        return None, 0
    hl = hybrid if isinstance(hybrid, (list, tuple)) else [hybrid]
    return (Hybrid * len(hl))(*[Hybrid(h["t_hyb"], h["window_s"], h["sigma_s"], int(h["taper"])) for h in hl]), len(hl)


STATIC_SCRATCH_BYTES = 64 << 20


def response_static(which, orb, hp, hc, sources, gen, order, fd_order=2, hybrid=None, out=None):
    """The response `which` (RESPONSE_FULL / _LFA / _HYBRID) without a workspace: the library's scratch is a static device
    array of STATIC_SCRATCH_BYTES, nothing is allocated by the call (ltdi_response_static).  out: dict of preallocated A, E,
    T [batch][ld] device tensors (allocated here if None: that allocation is the caller's, not the library's).  Calls that
    overlap on the GPU race on the shared array; LtdiError(EWORKSPACE) if the problem does not fit."""
    hp, hc = _dev_f64(hp, "hp"), _dev_f64(hc, "hc")
    if hp.dim() == 1:
        hp, hc = hp[None], hc[None]
    batch, ld = hp.shape
    assert hc.shape == hp.shape
    src_ptr, keep = _sources(sources)
    assert keep.shape[0] == batch, "one (beta, lambda, psi) per source"
    harr, nh = _hybrid_array(hybrid)
    if out is None:
        out = {c: torch.empty(batch, ld, dtype=torch.float64, device=hp.device) for c in "AET"}
    with torch.cuda.device(hp.device):
        rc = lib().ltdi_response_static(which, orb.handle, hp.data_ptr(), hc.data_ptr(), ld, batch, src_ptr, gen, order, fd_order,
                                        harr, nh, out["A"].data_ptr(), out["E"].data_ptr(), out["T"].data_ptr(), _stream())
    _check("ltdi_response_static", rc)
    return out


class HostPipeline:
    """End-to-end call with HOST buffers (ltdi_response_host): pinned strain in, pinned A, E, T out.

    depth = 1: every call is enqueued on the current stream.  depth > 1: successive calls rotate over `depth`
    slots, each with its own stream, device scratch and pinned outputs, so that the device->host copy of one call
    overlaps the host->device copy and the kernels of the next (PCIe is full duplex).  run() returns the slot's
    pinned A, E, T, valid after synchronize() (or once the slot is reused, after its event)."""

    def __init__(self, orb, batch, ld, depth=1):
        self.orb, self.batch, self.ld, self.depth = orb, batch, ld, int(depth)
        nbytes = C.c_size_t()
        _check("ltdi_host_scratch_bytes", lib().ltdi_host_scratch_bytes(ld, batch, C.byref(nbytes)))
        self.slots = []
        for _ in range(self.depth):
            slot = {"scratch": torch.empty(nbytes.value // 8, dtype=torch.float64, device=orb.device),
                    "out": tuple(torch.empty(batch, ld, dtype=torch.float64).pin_memory() for _ in range(3)),
                    "stream": torch.cuda.Stream(device=orb.device) if self.depth > 1 else None,
                    "event": None}
            self.slots.append(slot)
        self.A, self.E, self.T = self.slots[0]["out"]
        self.calls = 0
        self.h2d_bytes = 2 * batch * ld * 8
        self.d2h_bytes = 3 * batch * ld * 8

    def run(self, which, hp_host, hc_host, sources, gen, order, fd_order=2, hybrid=None):
        assert hp_host.dtype == torch.float64 and not hp_host.is_cuda and hp_host.is_contiguous()
        src_ptr, keep = _sources(sources)
        harr, nh = _hybrid_array(hybrid)
        slot = self.slots[self.calls % self.depth]
        self.calls += 1
        A, E, T = slot["out"]
        with torch.cuda.device(self.orb.device):
            if slot["stream"] is None:
                stream = _stream()
            else:
                if slot["event"] is not None:
                    slot["event"].synchronize()          # the slot's previous results have reached the host
                slot["stream"].wait_stream(torch.cuda.current_stream())   # orbit tables etc. of the caller
                stream = slot["stream"].cuda_stream
                # tensors allocated on another stream and read by the slot's stream: tell the caching allocator, so that
                # dropping the Orbits object while a call is in flight cannot hand their memory out again
                self.orb.tables.record_stream(slot["stream"])
                if self.orb._anchors is not None:
                    self.orb._anchors.record_stream(slot["stream"])
                slot["scratch"].record_stream(slot["stream"])
            rc = lib().ltdi_response_host(which, self.orb.handle, hp_host.data_ptr(), hc_host.data_ptr(), self.ld,
                                          self.batch, src_ptr, gen, order, fd_order, harr, nh, A.data_ptr(),
                                          E.data_ptr(), T.data_ptr(), slot["scratch"].data_ptr(),
                                          slot["scratch"].numel() * 8, stream)
            if slot["stream"] is not None:
                slot["event"] = torch.cuda.Event()
                slot["event"].record(slot["stream"])
        _check("ltdi_response_host", rc)
        return A, E, T

    def join(self):
        """Make the current stream wait for every call in flight (depth > 1)."""
        for slot in self.slots:
            if slot["stream"] is not None:
                torch.cuda.current_stream().wait_stream(slot["stream"])

    def synchronize(self):
        for slot in self.slots:
            if slot["stream"] is not None:
                slot["stream"].synchronize()
            else:
                torch.cuda.current_stream().synchronize()


class NoiseDesc(C.Structure):
    _fields_ = [("arm_m", C.c_double), ("t_obs_yr", C.c_double), ("gen", C.c_int32), ("galactic", C.c_int32)]


class Overlap:
    """FFT of A, E, T -> noise-weighted inner products, overlap, mismatch, SNR (Eqs. 5.1, 5.2, 6.1)
    of two responses of the same sources.  Owns the transform plan (lengths, chunking) and its device scratch; the Fourier transform is the library's own (csrc/fft.cuh)."""

    def __init__(self, n, ld, batch, device="cuda:0"):
        self.n, self.ld, self.batch, self.device = int(n), int(ld), int(batch), torch.device(device)
        handle, nbytes = C.c_void_p(), C.c_size_t()
        with torch.cuda.device(self.device):
            _check("ltdi_overlap_create", lib().ltdi_overlap_create(self.n, self.ld, self.batch, C.byref(handle),
                                                                    C.byref(nbytes)))
        self.handle = handle
        self.work = torch.empty((nbytes.value + 7) // 8, dtype=torch.float64, device=self.device)
        self.nf = self.n // 2 + 1
        self.out = torch.empty(self.batch, 3, 5, dtype=torch.float64, device=self.device)
        self.snr = torch.empty(self.batch, 3, dtype=torch.float64, device=self.device)

    def psd(self, dt, gen, arm_m=ARM_M, t_obs_yr=1.0, galactic=True):
        """[2][nf] device tensor: S_n^{A,E}, S_n^T on f_k = k / (n dt), Eqs. (2.10)-(2.13)."""
        d = NoiseDesc(float(arm_m), float(t_obs_yr), int(gen), int(bool(galactic)))
        psd = torch.empty(2, self.nf, dtype=torch.float64, device=self.device)
        with torch.cuda.device(self.device):
            _check("ltdi_noise_psd", lib().ltdi_noise_psd(C.byref(d), 1.0 / (self.n * float(dt)), self.nf,
                                                          psd.data_ptr(), _stream()))
        return psd

    def products(self, a, b, dt, psd, fmin, fmax):
        """a, b: dicts with device tensors A, E, T [batch][ld].  Returns (out [batch][3][5], snr [batch][3]):
        snr columns = rho_a, rho_b (6.1), ln L of (D4)."""
        t = [_dev_f64(x[c], c) for x in (a, b) for c in "AET"]
        for x in t:
            assert x.shape == (self.batch, self.ld) or (self.batch == 1 and x.numel() == self.ld)
        with torch.cuda.device(self.device):
            rc = lib().ltdi_overlap_products(self.handle, *[x.data_ptr() for x in t], float(dt), psd.data_ptr(),
                                             float(fmin), float(fmax), self.out.data_ptr(), self.snr.data_ptr(),
                                             self.work.data_ptr(), self.work.numel() * 8, _stream())
        _check("ltdi_overlap_products", rc)
        return self.out, self.snr

    def __del__(self):
        h, self.handle = getattr(self, "handle", None), None
        if h and _lib is not None:
            _lib.ltdi_overlap_destroy(h)


def fp64_probe(blocks=148 * 8, iters=2000, repeats=5, device="cuda:0"):
    """Measured DFMA issue rate [DFMA/s] of the device (register-resident chains, CUDA events)."""
    out = torch.empty(blocks * 256, dtype=torch.float64, device=device)
    n = C.c_double()
    best = 0.0
    with torch.cuda.device(out.device):
        for _ in range(repeats + 1):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            _check("ltdi_fp64_probe", lib().ltdi_fp64_probe(out.data_ptr(), blocks, iters, _stream(), C.byref(n)))
            e1.record()
            e1.synchronize()
            best = max(best, n.value / (e0.elapsed_time(e1) * 1e-3))
    return best
