"""ctypes binding of include/mcdc.h: argument marshalling only.

PyTorch provides the device workspace (a uint8 CUDA tensor) and the stream; nothing
else.  Importing works without a GPU (so the symbol test can run); any compute call
without a CUDA device or without the built extension raises.
"""
import ctypes as C
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "csrc", "libmcdc_b200.so")

COUNTER_NAMES = ("source", "flights", "segments", "collisions", "scatters", "captures",
                 "fissions", "secondaries", "crossings", "reflections", "leaks", "census",
                 "comb_in", "comb_out", "lost", "fingerprint")
STATUS = {0: "MCDC_OK", 1: "MCDC_EINVAL", 2: "MCDC_ENOMEM", 3: "MCDC_ECUDA", 4: "MCDC_ESTATE",
          5: "MCDC_EOVERFLOW", 6: "MCDC_ELOST"}

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


class McdcError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class Materials(C.Structure):
    _fields_ = [("n_mat", C.c_int32), ("n_group", C.c_int32), ("sigma_t", _dp), ("sigma_c", _dp),
                ("sigma_f", _dp), ("nu", _dp), ("sigma_s", _dp), ("chi", _dp), ("speed", _dp)]


class Geometry(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("xs", _dp), ("ys", _dp),
                ("zs", _dp), ("mat_outer", _ip), ("mat_inner", _ip), ("radius", _dp),
                ("bc", C.c_int32 * 6)]


class Source(C.Structure):
    _fields_ = [("kind", C.c_int32), ("lo", C.c_double * 3), ("hi", C.c_double * 3),
                ("isotropic", C.c_int32), ("dir", C.c_double * 3), ("group_pdf", _dp),
                ("t0", C.c_double)]


class TallyMesh(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("nt", C.c_int32),
                ("xs", _dp), ("ys", _dp), ("zs", _dp), ("ts", _dp), ("time_crossing", C.c_int32)]


class Census(C.Structure):
    _fields_ = [("n_census", C.c_int32), ("t_census", _dp), ("comb_target", C.c_uint64)]


class RunParams(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("n_hist_per_batch", C.c_uint64), ("n_batch", C.c_uint32),
                ("bank_capacity_factor", C.c_double)]


class Counters(C.Structure):
    _fields_ = [(n, C.c_uint64) for n in COUNTER_NAMES]


EXPORTS = ("mcdc_problem_create", "mcdc_workspace_bytes", "mcdc_run", "mcdc_tally_size",
           "mcdc_tally_read", "mcdc_counters_read", "mcdc_run_stats", "mcdc_kernel_path", "mcdc_profile",
           "mcdc_profile_read", "mcdc_replica_layout", "mcdc_replica_commit", "mcdc_set_csg", "mcdc_set_surface_motion", "mcdc_set_eigenvalue", "mcdc_keff_read", "mcdc_set_implicit_capture", "mcdc_set_delayed", "mcdc_set_source_window", "mcdc_batch_stats_noalloc", "mcdc_problem_destroy",
           "mcdc_last_error")

_lib = None


def load_library():
    """Loads csrc/libmcdc_b200.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2305_07636_b200.build` "
                          "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.mcdc_problem_create.argtypes = [C.POINTER(Materials), C.POINTER(Geometry), C.POINTER(Source),
                                      C.POINTER(TallyMesh), C.POINTER(Census), C.POINTER(vp)]
    L.mcdc_workspace_bytes.argtypes = [vp, C.POINTER(RunParams)]
    L.mcdc_workspace_bytes.restype = C.c_size_t
    L.mcdc_run.argtypes = [vp, C.POINTER(RunParams), vp, C.c_size_t, vp]
    L.mcdc_tally_size.argtypes = [vp]
    L.mcdc_tally_size.restype = C.c_size_t
    L.mcdc_tally_read.argtypes = [vp, C.c_int, vp, C.c_size_t, C.c_int]
    L.mcdc_counters_read.argtypes = [vp, C.c_uint32, C.c_int32, C.POINTER(Counters)]
    L.mcdc_run_stats.argtypes = [vp, C.POINTER(C.c_uint64), C.POINTER(C.c_uint64)]
    L.mcdc_kernel_path.argtypes = [vp, C.POINTER(C.c_int)]
    L.mcdc_profile.argtypes = [vp, C.c_int]
    L.mcdc_profile_read.argtypes = [vp, C.c_int, _dp, C.POINTER(C.c_uint64)]
    L.mcdc_replica_layout.argtypes = [vp] + [C.POINTER(C.c_size_t)] * 4
    L.mcdc_replica_commit.argtypes = [vp, C.c_uint32]
    L.mcdc_set_csg.argtypes = [vp, C.c_int32, _dp, C.c_int32, _ip, _ip]
    L.mcdc_set_surface_motion.argtypes = [vp, C.c_int32, _dp, _dp]
    L.mcdc_set_eigenvalue.argtypes = [vp, C.c_int32, C.c_int32, C.c_double]
    L.mcdc_keff_read.argtypes = [vp, C.c_uint32, _dp, C.c_size_t]
    L.mcdc_set_implicit_capture.argtypes = [vp, C.c_double, C.c_double]
    L.mcdc_set_delayed.argtypes = [vp, C.c_int32, _dp, _dp, _dp]
    L.mcdc_set_source_window.argtypes = [vp, C.c_double]
    L.mcdc_batch_stats_noalloc.argtypes = [vp, C.c_uint32, C.c_size_t, C.c_double, vp, vp, vp]
    L.mcdc_problem_destroy.argtypes = [vp]
    L.mcdc_problem_destroy.restype = None
    L.mcdc_last_error.restype = C.c_char_p
    _lib = L
    return L


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _pd(a):
    return a.ctypes.data_as(_dp)


NOALLOC_MAX_BINS = 1 << 20   # MCDC_NOALLOC_MAX_BINS of include/mcdc.h


def batch_stats_noalloc(batches, n_hist_per_batch, mean, stderr=None, stream=None):
    """mcdc_batch_stats_noalloc: mean (and standard error) over the rows of `batches` ([n_batch][n] float64 CUDA
    tensor of raw batch tallies) into the caller's CUDA tensors `mean` / `stderr` (n float64 each).  The library
    call allocates nothing and does not synchronise; the tensors are the caller's."""
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("no CUDA device: this path has no CPU fallback")
    L = load_library()
    for t in (batches, mean) + (() if stderr is None else (stderr,)):
        if not (t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()):
            raise ValueError("contiguous float64 CUDA tensors expected")
    if batches.dim() != 2 or mean.numel() != batches.shape[1] or (stderr is not None and stderr.numel() != batches.shape[1]):
        raise ValueError("batches [n_batch][n], mean [n], stderr [n]")
    s = torch.cuda.current_stream() if stream is None else stream
    rc = L.mcdc_batch_stats_noalloc(C.c_void_p(batches.data_ptr()), int(batches.shape[0]), int(batches.shape[1]),
                                    float(n_hist_per_batch), C.c_void_p(mean.data_ptr()),
                                    C.c_void_p(stderr.data_ptr()) if stderr is not None else None,
                                    C.c_void_p(s.cuda_stream))
    if rc != 0:
        raise McdcError(rc, L.mcdc_last_error().decode())


class Problem:
    """mcdc_problem handle built from a config dict (see mcdc_inputs)."""

    def __init__(self, cfg):
        L = self._L = load_library()
        m, g, s, t, c = (cfg[k] for k in ("materials", "geometry", "source", "tally", "census"))
        keep = {}
        mat = Materials()
        st = _d(m["sigma_t"])
        mat.n_mat, mat.n_group = st.shape
        for k in ("sigma_t", "sigma_c", "sigma_f", "nu", "sigma_s", "chi", "speed"):
            keep["m" + k] = _d(m[k]); setattr(mat, k, _pd(keep["m" + k]))
        geo = Geometry()
        geo.nx, geo.ny, geo.nz = len(g["xs"]) - 1, len(g["ys"]) - 1, len(g["zs"]) - 1
        for k in ("xs", "ys", "zs", "radius"):
            keep["g" + k] = _d(g[k]); setattr(geo, k, _pd(keep["g" + k]))
        for k in ("mat_outer", "mat_inner"):
            keep[k] = _i(g[k]); setattr(geo, k, keep[k].ctypes.data_as(_ip))
        if keep["mat_outer"].shape != (geo.nz, geo.ny, geo.nx):
            raise ValueError("mat_outer must have shape [nz][ny][nx]")
        geo.bc = (C.c_int32 * 6)(*[int(b) for b in g["bc"]])
        src = Source()
        src.kind = int(s["kind"]); src.isotropic = int(s["isotropic"]); src.t0 = float(s["t0"])
        src.lo = (C.c_double * 3)(*map(float, s["lo"])); src.hi = (C.c_double * 3)(*map(float, s["hi"]))
        src.dir = (C.c_double * 3)(*map(float, s["dir"]))
        keep["pdf"] = _d(s["group_pdf"]); src.group_pdf = _pd(keep["pdf"])
        tal = TallyMesh()
        tal.nx, tal.ny, tal.nz, tal.nt = (len(t[k]) - 1 for k in ("txs", "tys", "tzs", "tts"))
        for k, f in (("txs", "xs"), ("tys", "ys"), ("tzs", "zs"), ("tts", "ts")):
            keep[k] = _d(t[k]); setattr(tal, f, _pd(keep[k]))
        tal.time_crossing = int(t.get("time_crossing", 0))
        cen = Census()
        keep["tc"] = _d(c["t_census"]) if len(c["t_census"]) else np.zeros(1)
        cen.n_census = len(c["t_census"]); cen.t_census = _pd(keep["tc"])
        cen.comb_target = int(c["comb_target"])
        h = C.c_void_p()
        rc = L.mcdc_problem_create(C.byref(mat), C.byref(geo), C.byref(src), C.byref(tal), C.byref(cen),
                                   C.byref(h))
        if rc != 0:
            raise McdcError(rc, L.mcdc_last_error().decode())
        self._h = h
        self.shape = (tal.nt, mat.n_group, tal.nz, tal.ny, tal.nx)
        if tal.time_crossing:       # [0] track-length block, [1] time-crossing block (one bin per upper time edge)
            self.shape = (2,) + self.shape
        self.n_steps = max(int(cen.n_census), 1)
        if s.get("t_end") is not None:
            self._check(L.mcdc_set_source_window(h, float(s["t_end"])))
        csg = cfg.get("csg")
        if csg:
            coef, rs, rm = _d(csg["coef"]), _i(csg["region_surf"]), _i(csg["region_mat"])
            if coef.ndim != 2 or coef.shape[1] != 10 or rs.ndim != 2 or rs.shape[1] != 8 or rm.shape != (rs.shape[0],):
                raise ValueError("csg: coef [n_surf][10], region_surf [n_region][8], region_mat [n_region]")
            self._check(L.mcdc_set_csg(h, coef.shape[0], _pd(coef), rs.shape[0], rs.ctypes.data_as(_ip), rm.ctypes.data_as(_ip)))
            mv = cfg.get("motion")
            if mv:
                tau, disp = _d(mv["tau"]), _d(mv["disp"])
                if disp.shape != (coef.shape[0], tau.size, 3):
                    raise ValueError("motion: tau [n_tau], disp [n_surf][n_tau][3]")
                self._check(L.mcdc_set_surface_motion(h, tau.size, _pd(tau), _pd(disp)))
        dn = cfg.get("delayed")
        if dn:
            nud, lam, chd = (_d(dn[k]) for k in ("nu_delayed", "decay", "chi_delayed"))
            J = lam.shape[-1]
            if nud.shape != (mat.n_mat, mat.n_group, J) or lam.shape != (mat.n_mat, J) or chd.shape != (mat.n_mat, J, mat.n_group):
                raise ValueError("delayed: nu_delayed [M][G][J], decay [M][J], chi_delayed [M][J][G]")
            self._check(L.mcdc_set_delayed(h, J, _pd(nud), _pd(lam), _pd(chd)))
        ic = cfg.get("implicit_capture")
        if ic:
            self._check(L.mcdc_set_implicit_capture(h, float(ic["w_roulette"]), float(ic["w_survive"])))
        e = cfg.get("eigenvalue")
        if e:
            self._check(L.mcdc_set_eigenvalue(h, int(e["n_inactive"]), int(e["n_active"]), float(e["k0"])))
            self.n_steps = int(e["n_inactive"]) + int(e["n_active"])
        self.run_params = dict(cfg["run"])
        self._ws = None

    def _check(self, rc):
        if rc != 0:
            raise McdcError(rc, self._L.mcdc_last_error().decode())

    def params(self, seed=None, n_hist_per_batch=None, n_batch=None, bank_capacity_factor=0.0):
        r = self.run_params
        rp = RunParams()
        rp.seed = int(r["seed"] if seed is None else seed)
        rp.n_hist_per_batch = int(r["n_hist_per_batch"] if n_hist_per_batch is None else n_hist_per_batch)
        rp.n_batch = int(r["n_batch"] if n_batch is None else n_batch)
        rp.bank_capacity_factor = float(bank_capacity_factor)
        return rp

    def workspace_bytes(self, rp):
        n = self._L.mcdc_workspace_bytes(self._h, C.byref(rp))
        if n == 0:
            raise McdcError(1, self._L.mcdc_last_error().decode())
        return n

    def run(self, seed=None, n_hist_per_batch=None, n_batch=None, bank_capacity_factor=0.0,
            stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: this path has no CPU fallback")
        rp = self.params(seed, n_hist_per_batch, n_batch, bank_capacity_factor)
        nbytes = self.workspace_bytes(rp)
        if self._ws is None or self._ws.numel() < nbytes:
            self._ws = None
            self._ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        s = torch.cuda.current_stream() if stream is None else stream
        self.n_batch = rp.n_batch
        self._check(self._L.mcdc_run(self._h, C.byref(rp), C.c_void_p(self._ws.data_ptr()),
                                     self._ws.numel(), C.c_void_p(s.cuda_stream)))
        return self

    def tally(self, which=0, pinned=False):
        """Host copy of the tally.  pinned=True reads into a page-locked buffer owned by this object
        (a true asynchronous DMA; the returned array is a view that the next pinned read overwrites)."""
        n = self._L.mcdc_tally_size(self._h)
        if pinned:
            import torch
            if getattr(self, "_pin", None) is None or self._pin.numel() != n:
                self._pin = torch.empty(n, dtype=torch.float64, pin_memory=True)
            out = self._pin.numpy()
        else:
            out = np.empty(n)
        self._check(self._L.mcdc_tally_read(self._h, int(which), out.ctypes.data_as(C.c_void_p), n, 0))
        return out.reshape(self.shape)

    def tally_device(self, which=0):
        import torch
        n = self._L.mcdc_tally_size(self._h)
        out = torch.empty(n, dtype=torch.float64, device="cuda")
        self._check(self._L.mcdc_tally_read(self._h, int(which), C.c_void_p(out.data_ptr()), n, 1))
        return out.view(self.shape)

    def counters(self, batch=0, step=-1):
        c = Counters()
        self._check(self._L.mcdc_counters_read(self._h, int(batch), int(step), C.byref(c)))
        return {n: int(getattr(c, n)) for n in COUNTER_NAMES}

    def replica_views(self):
        """Views of the workspace tensor over (sum x .. sum x^2) as float64 and the counters as int64:
        what a sum all-reduce over the replicas acts on, in place (include/mcdc.h mcdc_replica_layout)."""
        import torch
        o1, o2, oc, nc = C.c_size_t(), C.c_size_t(), C.c_size_t(), C.c_size_t()
        self._check(self._L.mcdc_replica_layout(self._h, C.byref(o1), C.byref(o2), C.byref(oc), C.byref(nc)))
        n = self._L.mcdc_tally_size(self._h)
        sums = self._ws[o1.value:o2.value + 8 * n].view(torch.float64)
        cnt = self._ws[oc.value:oc.value + nc.value].view(torch.int64)
        return sums, cnt

    def replica_commit(self, n_ranks):
        self._check(self._L.mcdc_replica_commit(self._h, int(n_ranks)))

    def k_cycle(self, batch=0):
        """Generation estimate of k of every cycle of a batch (eigenvalue mode)."""
        out = np.empty(self.n_steps)
        self._check(self._L.mcdc_keff_read(self._h, int(batch), _pd(out), out.size))
        return out

    def stats(self):
        it, la = C.c_uint64(), C.c_uint64()
        self._check(self._L.mcdc_run_stats(self._h, C.byref(it), C.byref(la)))
        return dict(iterations=it.value, launches=la.value)

    def profile(self, enable=True):
        self._check(self._L.mcdc_profile(self._h, int(enable)))

    def kernel_path(self):
        """'pool' (one persistent launch per census step) or 'events' (per-event kernels)."""
        v = C.c_int()
        self._check(self._L.mcdc_kernel_path(self._h, C.byref(v)))
        return "pool" if v.value else "events"

    def profile_read(self):
        out = {}
        names = ("k_pool", "k_collide") if self.kernel_path() == "pool" else ("k_flight", "k_collide")
        for k, name in enumerate(names):
            ms, n = C.c_double(), C.c_uint64()
            self._check(self._L.mcdc_profile_read(self._h, k, C.byref(ms), C.byref(n)))
            out[name] = dict(ms=ms.value, launches=n.value)
        return out

    def close(self):
        if getattr(self, "_h", None):
            self._L.mcdc_problem_destroy(self._h)
            self._h = None
        self._ws = None
        self._pin = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
