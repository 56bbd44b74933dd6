"""ctypes binding of the oracle (argument marshalling only).  TEST INFRASTRUCTURE ONLY."""
import ctypes as C

import numpy as np

from .build import build

COUNTER_NAMES = ("source", "flights", "segments", "collisions", "scatters", "captures",
                 "fissions", "secondaries", "crossings", "reflections", "leaks", "census",
                 "comb_in", "comb_out", "lost", "fingerprint")

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class _Input(C.Structure):
    _fields_ = [
        ("n_mat", C.c_int32), ("n_group", C.c_int32),
        ("sigma_t", _dp), ("sigma_c", _dp), ("sigma_f", _dp), ("nu", _dp), ("sigma_s", _dp),
        ("chi", _dp), ("speed", _dp),
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("xs", _dp), ("ys", _dp), ("zs", _dp),
        ("mat_outer", _ip), ("mat_inner", _ip), ("radius", _dp), ("bc", C.c_int32 * 6),
        ("src_kind", C.c_int32), ("src_lo", C.c_double * 3), ("src_hi", C.c_double * 3),
        ("src_isotropic", C.c_int32), ("src_dir", C.c_double * 3), ("src_group_pdf", _dp),
        ("src_t0", C.c_double),
        ("tnx", C.c_int32), ("tny", C.c_int32), ("tnz", C.c_int32), ("tnt", C.c_int32),
        ("txs", _dp), ("tys", _dp), ("tzs", _dp), ("tts", _dp), ("time_crossing", C.c_int32),
        ("n_census", C.c_int32), ("t_census", _dp), ("comb_target", C.c_uint64),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.oracle_create.argtypes = [C.POINTER(_Input), C.POINTER(C.c_void_p)]
        L.oracle_destroy.argtypes = [C.c_void_p]
        L.oracle_destroy.restype = None
        L.oracle_run.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_uint32]
        L.oracle_tally_size.argtypes = [C.c_void_p]
        L.oracle_tally_size.restype = C.c_size_t
        L.oracle_tally_read.argtypes = [C.c_void_p, C.c_int, _dp, C.c_size_t]
        L.oracle_counters_read.argtypes = [C.c_void_p, C.c_uint32, C.c_int32, C.POINTER(C.c_uint64)]
        L.oracle_set_eigenvalue.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_double]
        L.oracle_keff_read.argtypes = [C.c_void_p, C.c_uint32, _dp, C.c_size_t]
        L.oracle_set_implicit_capture.argtypes = [C.c_void_p, C.c_double, C.c_double]
        L.oracle_comb_weighted.argtypes = [C.c_uint64, C.c_uint64, C.c_double, _dp, C.POINTER(C.c_uint64), _dp]
        L.oracle_set_source_window.argtypes = [C.c_void_p, C.c_double]
        L.oracle_set_delayed.argtypes = [C.c_void_p, C.c_int32, _dp, _dp, _dp]
        L.oracle_n_steps.argtypes = [C.c_void_p]
        L.oracle_n_steps.restype = C.c_uint64
        L.oracle_philox4x32_10.argtypes = [C.POINTER(C.c_uint32)] * 3
        L.oracle_philox4x32_10.restype = None
        L.oracle_uniform52.argtypes = [C.c_uint32, C.c_uint32]
        L.oracle_uniform52.restype = C.c_double
        L.oracle_log.argtypes = [C.c_double]
        L.oracle_log.restype = C.c_double
        L.oracle_sincos2pi.argtypes = [C.c_double, _dp, _dp]
        L.oracle_sincos2pi.restype = None
        L.oracle_set_csg.argtypes = [C.c_void_p, C.c_int32, _dp, C.c_int32, _ip, _ip]
        L.oracle_set_surface_motion.argtypes = [C.c_void_p, C.c_int32, _dp, _dp]
        L.oracle_quadric_distance.argtypes = [_dp] + [C.c_double] * 7
        L.oracle_quadric_distance.restype = C.c_double
        L.oracle_isotropic.argtypes = [C.c_double, C.c_double, _dp]
        L.oracle_isotropic.restype = None
        L.oracle_cyl_distance.argtypes = [C.c_double] * 7 + [C.c_int]
        L.oracle_cyl_distance.restype = C.c_double
        L.oracle_march.argtypes = [_dp, C.c_int32, _dp, C.c_int32, _dp, C.c_int32, _dp, C.c_int32,
                                   _dp, C.c_double, _dp, C.c_double, C.c_double,
                                   C.POINTER(C.c_int64), _dp, C.c_int64]
        L.oracle_march.restype = C.c_int64
        L.oracle_comb_indices.argtypes = [C.c_uint64, C.c_uint64, C.c_double, C.POINTER(C.c_uint64)]
        L.oracle_comb_indices.restype = None
        _lib = L
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _pd(a):
    return a.ctypes.data_as(_dp)


class Oracle:
    """Problem handle built from a mcdc_inputs config dict."""

    def __init__(self, cfg):
        L = lib()
        m, g, s, t, c = (cfg[k] for k in ("materials", "geometry", "source", "tally", "census"))
        keep = self._keep = {}
        inp = _Input()
        st = _d(m["sigma_t"])
        inp.n_mat, inp.n_group = st.shape
        for k in ("sigma_t", "sigma_c", "sigma_f", "nu", "sigma_s", "chi", "speed"):
            keep[k] = _d(m[k]); setattr(inp, k, _pd(keep[k]))
        for k in ("xs", "ys", "zs", "radius"):
            keep[k] = _d(g[k]); setattr(inp, k, _pd(keep[k]))
        inp.nx, inp.ny, inp.nz = (len(g["xs"]) - 1, len(g["ys"]) - 1, len(g["zs"]) - 1)
        for k in ("mat_outer", "mat_inner"):
            keep[k] = _i(g[k]); setattr(inp, k, keep[k].ctypes.data_as(_ip))
        assert keep["mat_outer"].shape == (inp.nz, inp.ny, inp.nx)
        inp.bc = (C.c_int32 * 6)(*[int(b) for b in g["bc"]])
        inp.src_kind = int(s["kind"])
        inp.src_lo = (C.c_double * 3)(*[float(v) for v in s["lo"]])
        inp.src_hi = (C.c_double * 3)(*[float(v) for v in s["hi"]])
        inp.src_isotropic = int(s["isotropic"])
        inp.src_dir = (C.c_double * 3)(*[float(v) for v in s["dir"]])
        keep["pdf"] = _d(s["group_pdf"]); inp.src_group_pdf = _pd(keep["pdf"])
        inp.src_t0 = float(s["t0"])
        for k in ("txs", "tys", "tzs", "tts"):
            keep[k] = _d(t[k]); setattr(inp, k, _pd(keep[k]))
        inp.tnx, inp.tny, inp.tnz, inp.tnt = (len(t[k]) - 1 for k in ("txs", "tys", "tzs", "tts"))
        inp.time_crossing = int(t.get("time_crossing", 0))
        keep["tc"] = _d(c["t_census"]) if len(c["t_census"]) else np.zeros(1)
        inp.n_census = len(c["t_census"]); inp.t_census = _pd(keep["tc"])
        inp.comb_target = int(c["comb_target"])
        h = C.c_void_p()
        rc = L.oracle_create(C.byref(inp), C.byref(h))
        if rc != 0:
            raise ValueError(f"oracle_create failed: {rc}")
        self._h = h
        self.G = int(inp.n_group)
        self.shape = (inp.tnt, inp.n_group, inp.tnz, inp.tny, inp.tnx)
        if inp.time_crossing:       # [0] track-length block, [1] time-crossing block (one bin per upper time edge)
            self.shape = (2,) + self.shape
        if cfg["source"].get("t_end") is not None:
            if L.oracle_set_source_window(h, float(cfg["source"]["t_end"])) != 0:
                raise ValueError("oracle_set_source_window failed")
        csg = cfg.get("csg")
        if csg:
            coef = _d(csg["coef"]); rs = _i(csg["region_surf"]); rm = _i(csg["region_mat"])
            if coef.ndim != 2 or coef.shape[1] != 10 or rs.ndim != 2 or rs.shape[1] != 8 or rm.shape != (rs.shape[0],):
                raise ValueError("csg: coef [n_surf][10], region_surf [n_region][8], region_mat [n_region]")
            if L.oracle_set_csg(h, coef.shape[0], _pd(coef), rs.shape[0], rs.ctypes.data_as(_ip), rm.ctypes.data_as(_ip)) != 0:
                raise ValueError("oracle_set_csg failed")
            mv = cfg.get("motion")
            if mv:
                tau = _d(mv["tau"]); disp = _d(mv["disp"])
                if disp.shape != (coef.shape[0], tau.size, 3):
                    raise ValueError("motion: tau [n_tau], disp [n_surf][n_tau][3]")
                if L.oracle_set_surface_motion(h, tau.size, _pd(tau), _pd(disp)) != 0:
                    raise ValueError("oracle_set_surface_motion failed")
        dn = cfg.get("delayed")
        if dn:
            nud, lam, chd = (np.ascontiguousarray(dn[k], dtype=np.float64) for k in ("nu_delayed", "decay", "chi_delayed"))
            J = lam.shape[-1]
            if nud.shape != (inp.n_mat, inp.n_group, J) or lam.shape != (inp.n_mat, J) or chd.shape != (inp.n_mat, J, inp.n_group):
                raise ValueError("delayed: nu_delayed [M][G][J], decay [M][J], chi_delayed [M][J][G]")
            if L.oracle_set_delayed(h, J, _pd(nud), _pd(lam), _pd(chd)) != 0:
                raise ValueError("oracle_set_delayed failed")
        ic = cfg.get("implicit_capture")
        if ic:
            if L.oracle_set_implicit_capture(h, float(ic["w_roulette"]), float(ic["w_survive"])) != 0:
                raise ValueError("oracle_set_implicit_capture failed")
        e = cfg.get("eigenvalue")
        if e:
            if L.oracle_set_eigenvalue(h, int(e["n_inactive"]), int(e["n_active"]), float(e["k0"])) != 0:
                raise ValueError("oracle_set_eigenvalue failed")
        self.n_steps = int(L.oracle_n_steps(h))
        self.run_params = dict(cfg["run"])

    def run(self, seed=None, n_hist_per_batch=None, n_batch=None):
        r = self.run_params
        seed = r["seed"] if seed is None else seed
        n = r["n_hist_per_batch"] if n_hist_per_batch is None else n_hist_per_batch
        b = r["n_batch"] if n_batch is None else n_batch
        rc = lib().oracle_run(self._h, int(seed), int(n), int(b))
        if rc != 0:
            raise RuntimeError(f"oracle_run failed: {rc}")
        self.n_batch = int(b)
        return self

    def tally(self, which=0):
        n = lib().oracle_tally_size(self._h)
        out = np.empty(n)
        rc = lib().oracle_tally_read(self._h, int(which), _pd(out), n)
        if rc != 0:
            raise RuntimeError("oracle_tally_read failed")
        return out.reshape(self.shape)

    def counters(self, batch=0, step=-1):
        out = (C.c_uint64 * 16)()
        rc = lib().oracle_counters_read(self._h, int(batch), int(step), out)
        if rc != 0:
            raise RuntimeError("oracle_counters_read failed")
        return dict(zip(COUNTER_NAMES, (int(v) for v in out)))

    def k_cycle(self, batch=0):
        """Generation estimate of k of every cycle of a batch (eigenvalue mode)."""
        out = np.empty(self.n_steps)
        if lib().oracle_keff_read(self._h, int(batch), _pd(out), out.size) != 0:
            raise RuntimeError("oracle_keff_read failed")
        return out

    def close(self):
        if getattr(self, "_h", None):
            lib().oracle_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
