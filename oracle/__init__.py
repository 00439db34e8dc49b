"""ctypes front end of the CPU oracle -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this package.  It imports nothing from paper_2505_09600_b200.

    from oracle import Oracle
    orc = Oracle("f80")          # long double parity reference ("f64": timed baseline)
    out = orc.response_full(orbit, hp, hc, sources, gen=20, order=31)

`orbit` is a plain dict {t0, dt, n, arm_m, R_m, period_s, alpha0, rot0, mode} (see
workloads.orbit_desc), `sources` an array [batch][3] of (beta, lambda, psi),
hp / hc arrays [batch][n] of float64.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

GEN_15, GEN_20 = 15, 20
ORBIT_STATIC_EQUALARM, ORBIT_KEPLERIAN, ORBIT_TABLES, ORBIT_KNOTS = 0, 1, 2, 3
TAPER_SIGMOID, TAPER_COSINE = 0, 1


class _OrbitDesc(C.Structure):
    _fields_ = [("t0", C.c_double), ("dt", C.c_double), ("n", C.c_int64), ("arm_m", C.c_double),
                ("R_m", C.c_double), ("period_s", C.c_double), ("alpha0", C.c_double),
                ("rot0", C.c_double), ("mode", C.c_int32)]


class _Source(C.Structure):
    _fields_ = [("beta", C.c_double), ("lam", C.c_double), ("psi", C.c_double)]


class _Chirp(C.Structure):
    _fields_ = [("t_c", C.c_double), ("mc_s", C.c_double), ("dist_m", C.c_double), ("cos_iota", C.c_double),
                ("phi_c", C.c_double), ("tau_cut", C.c_double), ("f_rd", C.c_double), ("tau_rd", C.c_double)]


CHIRP_KEYS = ("t_c", "mc_s", "dist_m", "cos_iota", "phi_c", "tau_cut", "f_rd", "tau_rd")


class _Hybrid(C.Structure):
    _fields_ = [("t_hyb", C.c_double), ("window_s", C.c_double), ("sigma_s", C.c_double),
                ("taper", C.c_int32)]


_dp = C.POINTER(C.c_double)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class Oracle:
    def __init__(self, precision="f80", threads=None):
        libs = _build.build()
        self.precision = precision
        self.lib = C.CDLL(libs[precision])
        self.lib.orc_hyb_time.restype = C.c_double
        self.lib.orc_lfa_fraction.restype = C.c_double
        self.lib.orc_interp.restype = C.c_double
        self.lib.orc_hyb_time.argtypes = [C.c_double] * 3
        self.lib.orc_lfa_fraction.argtypes = [C.c_double] * 3
        self.lib.orc_interp.argtypes = [_dp, C.c_int64, C.c_int64, C.c_double, C.c_double, C.c_int]
        if threads is not None:
            os.environ["OMP_NUM_THREADS"] = str(int(threads))

    # -- helpers -------------------------------------------------------------------------
    @staticmethod
    def _desc(orbit):
        return _OrbitDesc(orbit["t0"], orbit["dt"], int(orbit["n"]), orbit["arm_m"], orbit["R_m"],
                          orbit["period_s"], orbit["alpha0"], orbit["rot0"], int(orbit["mode"]))

    @staticmethod
    def _tables(orbit):
        if int(orbit["mode"]) == ORBIT_KNOTS:   # a numerical orbit file: knots [3][3][nk] and {t0, dt, nk, order} of the knot grid
            K = _f64(orbit["knots"])
            assert K.ndim == 3 and K.shape[:2] == (3, 3)
            return K, _f64([orbit["knot_t0"], orbit["knot_dt"], K.shape[2], orbit["knot_order"]])
        if int(orbit["mode"]) != ORBIT_TABLES:
            return None, None
        R = _f64(orbit["R_table"])   # [3][3][n]
        L = _f64(orbit["L_table"])   # [6][n]
        assert R.shape == (3, 3, orbit["n"]) and L.shape == (6, orbit["n"])
        return R, L

    @staticmethod
    def _sources(sources):
        s = np.atleast_2d(_f64(sources))
        arr = (_Source * len(s))()
        for i, (b, l, p) in enumerate(s):
            arr[i] = _Source(b, l, p)
        return arr, len(s)

    def num_threads(self):
        return self.lib.orc_num_threads()

    def mant_dig(self):
        return self.lib.orc_real_mant_dig()

    def margins(self, orbit, gen, order, fd_order=0):
        lo, hi = C.c_int64(), C.c_int64()
        d = self._desc(orbit)
        rc = self.lib.orc_margins(C.byref(d), gen, order, fd_order, C.byref(lo), C.byref(hi))
        assert rc == 0
        return lo.value, hi.value

    def link_margins(self, orbit, order, fd_order=0):
        lo, hi = C.c_int64(), C.c_int64()
        d = self._desc(orbit)
        rc = self.lib.orc_link_margins(C.byref(d), order, fd_order, C.byref(lo), C.byref(hi))
        assert rc == 0
        return lo.value, hi.value

    def hyb_time(self, f_hyb, mchirp_s, t_c):
        return self.lib.orc_hyb_time(f_hyb, mchirp_s, t_c)

    def lfa_fraction(self, f_hyb, f_min, f_max):
        return self.lib.orc_lfa_fraction(f_hyb, f_min, f_max)

    def lagrange_weights(self, eps, order):
        w = np.zeros(order + 1)
        self.lib.orc_lagrange_weights(C.c_double(eps), order, _ptr(w))
        return w

    def interp(self, x, n, d, dt, order):
        x = _f64(x)
        return self.lib.orc_interp(_ptr(x), len(x), int(n), float(d), float(dt), order)

    def stencil(self, x, dt, fd_order, which):
        x = _f64(x)
        out = np.zeros_like(x)
        self.lib.orc_stencil(_ptr(x), C.c_int64(len(x)), C.c_double(dt), fd_order, which, _ptr(out))
        return out

    def source_frame(self, beta, lam, psi):
        out = np.zeros(11)
        s = _Source(beta, lam, psi)
        self.lib.orc_source_frame(C.byref(s), _ptr(out))
        return {"k": out[0:3], "u": out[3:6], "v": out[6:9], "c2": out[9], "s2": out[10]}

    def orbit_tables(self, orbit, nb=0, ne=None):
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        R, nh, L = np.zeros((3, 3, ln)), np.zeros((6, 3, ln)), np.zeros((6, ln))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_orbit_tables(C.byref(d), _ptr(Rt), _ptr(Lt), C.c_int64(nb), C.c_int64(ne),
                                       _ptr(R), _ptr(nh), _ptr(L))
        assert rc == 0
        return R, nh, L

    def orbit_tables_split(self, orbit, nb=0, ne=None):
        """n_l and L_l as hi + lo doubles (the working precision of this build split in two)."""
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        nh, nl, Lh, Ll = np.zeros((6, 3, ln)), np.zeros((6, 3, ln)), np.zeros((6, ln)), np.zeros((6, ln))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_orbit_tables_split(C.byref(d), _ptr(Rt), _ptr(Lt), C.c_int64(nb), C.c_int64(ne),
                                             _ptr(nh), _ptr(nl), _ptr(Lh), _ptr(Ll))
        assert rc == 0
        return nh, nl, Lh, Ll

    def michelson_from_links(self, orbit, y, gen, order):
        """X, Y, Z [3][n] of Eq. (2.7) / (2.8) from caller-supplied link series y [6][n]."""
        y = _f64(y)
        assert y.shape == (6, orbit["n"])
        out = np.zeros((3, orbit["n"]))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_michelson_from_links(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(y), C.c_int(gen), C.c_int(order),
                                               _ptr(out))
        assert rc == 0
        return out

    def sagnac_from_links(self, orbit, y, gen, order):
        """O15: alpha, beta, gamma [3][n] from caller-supplied link series y [6][n]."""
        y = _f64(y)
        assert y.shape == (6, orbit["n"])
        out = np.zeros((3, orbit["n"]))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_sagnac_from_links(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(y), C.c_int(gen), C.c_int(order), _ptr(out))
        assert rc == 0
        return out

    def antenna(self, orbit, source, n):
        out = np.zeros((6, 3))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        s = _Source(*[float(x) for x in source])
        self.lib.orc_antenna(C.byref(d), _ptr(Rt), _ptr(Lt), C.byref(s), C.c_int64(n), _ptr(out))
        return out  # rows: link; cols: F+, Fx, k.n

    def hybrid_weights(self, hyb, t):
        t = _f64(t)
        a, b = np.zeros_like(t), np.zeros_like(t)
        h = _Hybrid(hyb["t_hyb"], hyb["window_s"], hyb["sigma_s"], int(hyb["taper"]))
        self.lib.orc_hybrid_weights(C.byref(h), _ptr(t), C.c_int64(len(t)), _ptr(a), _ptr(b))
        return a, b

    # -- responses -----------------------------------------------------------------------
    def _run(self, which, orbit, hp, hc, sources, gen, order, fd_order, hyb, nb, ne, want):
        hp, hc = np.atleast_2d(_f64(hp)), np.atleast_2d(_f64(hc))
        batch, ld = hp.shape
        assert hc.shape == hp.shape and ld >= orbit["n"]
        src, ns = self._sources(sources)
        assert ns == batch
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        out = {"A": np.zeros((batch, ln)), "E": np.zeros((batch, ln)), "T": np.zeros((batch, ln))}
        out["XYZ"] = np.zeros((3, batch, ln)) if "XYZ" in want else None
        out["y"] = np.zeros((6, batch, ln)) if "y" in want else None
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        head = [C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(hp), _ptr(hc), C.c_int64(ld), C.c_int64(batch),
                src, C.c_int(gen), C.c_int(order)]
        tail = [C.c_int64(nb), C.c_int64(ne), _ptr(out["A"]), _ptr(out["E"]), _ptr(out["T"]),
                _ptr(out["XYZ"]), _ptr(out["y"])]
        if which == "full":
            rc = self.lib.orc_response_full(*head, *tail)
        elif which == "sagnac":
            rc = self.lib.orc_response_full_sagnac(*head, *tail)
        elif which == "lfa":
            rc = self.lib.orc_response_lfa(*head, C.c_int(fd_order), *tail)
        else:
            hl = hyb if isinstance(hyb, (list, tuple)) else [hyb]
            harr = (_Hybrid * len(hl))()
            for i, h in enumerate(hl):
                harr[i] = _Hybrid(h["t_hyb"], h["window_s"], h["sigma_s"], int(h["taper"]))
            rc = self.lib.orc_response_hybrid(*head, C.c_int(fd_order), harr, C.c_int64(len(hl)), *tail)
        if rc != 0:
            raise ValueError(f"oracle {which}: status {rc}")
        return out

    def response_full(self, orbit, hp, hc, sources, gen, order, nb=0, ne=None, want=("XYZ", "y")):
        return self._run("full", orbit, hp, hc, sources, gen, order, 0, None, nb, ne, want)

    def response_full_sagnac(self, orbit, hp, hc, sources, gen, order, nb=0, ne=None, want=("XYZ", "y")):
        """O15: the full response in the Sagnac combinations; out["XYZ"] holds alpha, beta, gamma."""
        return self._run("sagnac", orbit, hp, hc, sources, gen, order, 0, None, nb, ne, want)

    def response_full_nested(self, orbit, hp, hc, sources, gen, order, nested_order=3, nb=0, ne=None, want=("XYZ", "y")):
        """the full response with properly nested TDI delays (O12); nested_order = Lagrange order of the
        light-time lookups at off-grid times."""
        hp, hc = np.atleast_2d(_f64(hp)), np.atleast_2d(_f64(hc))
        batch, ld = hp.shape
        src, ns = self._sources(sources)
        assert ns == batch and ld >= orbit["n"]
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        out = {"A": np.zeros((batch, ln)), "E": np.zeros((batch, ln)), "T": np.zeros((batch, ln))}
        out["XYZ"] = np.zeros((3, batch, ln)) if "XYZ" in want else None
        out["y"] = np.zeros((6, batch, ln)) if "y" in want else None
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_response_full_nested(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(hp), _ptr(hc), C.c_int64(ld),
                                               C.c_int64(batch), src, C.c_int(gen), C.c_int(order), C.c_int(nested_order),
                                               C.c_int64(nb), C.c_int64(ne), _ptr(out["A"]), _ptr(out["E"]), _ptr(out["T"]),
                                               _ptr(out["XYZ"]), _ptr(out["y"]))
        if rc != 0:
            raise ValueError(f"oracle full_nested: status {rc}")
        return out

    def michelson_nested_from_links(self, orbit, y, gen, order, nested_order=3):
        """X, Y, Z [3][n] with nested delays (O12) from caller-supplied link series y [6][n]."""
        y = _f64(y)
        assert y.shape == (6, orbit["n"])
        out = np.zeros((3, orbit["n"]))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_michelson_nested_from_links(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(y), C.c_int(gen), C.c_int(order),
                                                      C.c_int(nested_order), _ptr(out))
        assert rc == 0
        return out

    @staticmethod
    def _chirps(params):
        arr = (_Chirp * len(params))()
        for i, p in enumerate(params):
            arr[i] = _Chirp(*[float(p[k]) for k in CHIRP_KEYS])
        return arr

    def waveform_chirp(self, params, t0, dt, n):
        """O13: the chirp + ringdown model sampled on t0 + i dt: hp, hc [batch][n] (rounded to double)."""
        hp, hc = np.zeros((len(params), n)), np.zeros((len(params), n))
        rc = self.lib.orc_waveform_chirp(self._chirps(params), C.c_int64(len(params)), C.c_double(t0), C.c_double(dt),
                                         C.c_int64(n), C.c_int64(n), _ptr(hp), _ptr(hc))
        if rc != 0:
            raise ValueError(f"oracle waveform_chirp: status {rc}")
        return hp, hc

    def waveform_ecc(self, tables, params, nharm, t0, dt, n):
        """O13b: the eccentric harmonic-sum model (tables [batch][7][nk], params [batch][6]) sampled on t0 + i dt."""
        tab, par = _f64(tables), _f64(params)
        batch, _, nk = tab.shape
        hp, hc = np.zeros((batch, n)), np.zeros((batch, n))
        rc = self.lib.orc_waveform_ecc(_ptr(tab), C.c_int64(nk), _ptr(par), C.c_int(nharm), C.c_int64(batch), C.c_double(t0),
                                       C.c_double(dt), C.c_int64(n), C.c_int64(n), _ptr(hp), _ptr(hc))
        if rc != 0:
            raise ValueError(f"oracle waveform_ecc: status {rc}")
        return hp, hc

    def response_full_chirp(self, orbit, params, sources, gen, order, nb=0, ne=None, want=("XYZ", "y")):
        """O13: Eq. (2.5) with the model evaluated at the retarded times, then O6 / O7."""
        batch = len(params)
        src, ns = self._sources(sources)
        assert ns == batch
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        out = {"A": np.zeros((batch, ln)), "E": np.zeros((batch, ln)), "T": np.zeros((batch, ln))}
        out["XYZ"] = np.zeros((3, batch, ln)) if "XYZ" in want else None
        out["y"] = np.zeros((6, batch, ln)) if "y" in want else None
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_response_full_chirp(C.byref(d), _ptr(Rt), _ptr(Lt), self._chirps(params), C.c_int64(batch), src,
                                              C.c_int(gen), C.c_int(order), C.c_int64(nb), C.c_int64(ne), _ptr(out["A"]),
                                              _ptr(out["E"]), _ptr(out["T"]), _ptr(out["XYZ"]), _ptr(out["y"]))
        if rc != 0:
            raise ValueError(f"oracle full_chirp: status {rc}")
        return out

    def response_lfa(self, orbit, hp, hc, sources, gen, order, fd_order, nb=0, ne=None,
                     want=("XYZ", "y")):
        return self._run("lfa", orbit, hp, hc, sources, gen, order, fd_order, None, nb, ne, want)

    def stencil3(self, x, dt, fd_order):
        x = _f64(x)
        out = np.zeros_like(x)
        self.lib.orc_stencil3(_ptr(x), C.c_int64(len(x)), C.c_double(dt), fd_order, _ptr(out))
        return out

    def margins_lfa_ext(self, orbit, gen, order, fd_order, terms=1):
        lo, hi = C.c_int64(), C.c_int64()
        d = self._desc(orbit)
        assert self.lib.orc_margins_lfa_ext(C.byref(d), gen, order, fd_order, terms, C.byref(lo), C.byref(hi)) == 0
        return lo.value, hi.value

    def response_lfa_ext(self, orbit, hp, hc, sources, gen, order, fd_order, terms=1, point=0, nb=0, ne=None,
                         want=("XYZ", "y")):
        """`terms` terms of Eq. (B4) about the expansion point (0 central, 1 backward, 2 forward)."""
        hp, hc = np.atleast_2d(_f64(hp)), np.atleast_2d(_f64(hc))
        batch, ld = hp.shape
        src, ns = self._sources(sources)
        assert ns == batch and ld >= orbit["n"]
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        out = {"A": np.zeros((batch, ln)), "E": np.zeros((batch, ln)), "T": np.zeros((batch, ln))}
        out["XYZ"] = np.zeros((3, batch, ln)) if "XYZ" in want else None
        out["y"] = np.zeros((6, batch, ln)) if "y" in want else None
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_response_lfa_ext(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(hp), _ptr(hc), C.c_int64(ld),
                                           C.c_int64(batch), src, C.c_int(gen), C.c_int(order), C.c_int(fd_order),
                                           C.c_int(terms), C.c_int(point), C.c_int64(nb), C.c_int64(ne), _ptr(out["A"]),
                                           _ptr(out["E"]), _ptr(out["T"]), _ptr(out["XYZ"]), _ptr(out["y"]))
        if rc != 0:
            raise ValueError(f"oracle lfa_ext: status {rc}")
        return out

    def margins_lfa6(self, orbit, gen, order, fd_order):
        lo, hi = C.c_int64(), C.c_int64()
        d = self._desc(orbit)
        assert self.lib.orc_margins_lfa6(C.byref(d), gen, order, fd_order, C.byref(lo), C.byref(hi)) == 0
        return lo.value, hi.value

    def response_lfa6(self, orbit, hp, hc, sources, gen, order, fd_order, nb=0, ne=None, want=("XYZ", "y")):
        """O14: all six LFA links and the Michelson variables of Eq. (B20) / (B30) (no link-reversal symmetry)."""
        hp, hc = np.atleast_2d(_f64(hp)), np.atleast_2d(_f64(hc))
        batch, ld = hp.shape
        src, ns = self._sources(sources)
        assert ns == batch and ld >= orbit["n"]
        ne = orbit["n"] if ne is None else ne
        ln = ne - nb
        out = {"A": np.zeros((batch, ln)), "E": np.zeros((batch, ln)), "T": np.zeros((batch, ln))}
        out["XYZ"] = np.zeros((3, batch, ln)) if "XYZ" in want else None
        out["y"] = np.zeros((6, batch, ln)) if "y" in want else None
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_response_lfa6(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(hp), _ptr(hc), C.c_int64(ld), C.c_int64(batch), src,
                                        C.c_int(gen), C.c_int(order), C.c_int(fd_order), C.c_int64(nb), C.c_int64(ne),
                                        _ptr(out["A"]), _ptr(out["E"]), _ptr(out["T"]), _ptr(out["XYZ"]), _ptr(out["y"]))
        if rc != 0:
            raise ValueError(f"oracle lfa6: status {rc}")
        return out

    def michelson_b20_from_links(self, orbit, y, gen, order, fd_order):
        """X, Y, Z [3][n] of Eq. (B20) / (B30) from caller-supplied link series y [6][n]."""
        y = _f64(y)
        assert y.shape == (6, orbit["n"])
        out = np.zeros((3, orbit["n"]))
        d = self._desc(orbit)
        Rt, Lt = self._tables(orbit)
        rc = self.lib.orc_michelson_b20_from_links(C.byref(d), _ptr(Rt), _ptr(Lt), _ptr(y), C.c_int(gen), C.c_int(order),
                                                   C.c_int(fd_order), _ptr(out))
        assert rc == 0
        return out

    def response_hybrid(self, orbit, hp, hc, sources, gen, order, fd_order, hyb, nb=0, ne=None,
                        want=("XYZ", "y")):
        return self._run("hybrid", orbit, hp, hc, sources, gen, order, fd_order, hyb, nb, ne, want)
