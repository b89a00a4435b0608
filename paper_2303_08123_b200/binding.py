"""Thin Python binding of the C ABI in include/ca.h (same names, argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libca_b200.so; PyTorch is used for device
memory (the workspace tensor) and streams.  There is NO CPU fallback: load() raises if the library
is missing, and ca_create fails without a CUDA device.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libca_b200.so")

CA_OK, CA_EINVAL, CA_EPROTO, CA_ESTATE, CA_ECUDA, CA_EOVERFLOW = 0, -1, -2, -3, -4, -5
CA_NCOUNT = 13
COUNT_NAMES = ("live", "doomed", "ready", "dead", "G1", "S", "G2", "M", "PA", "PN", "QA", "QN", "occupied")
INIT_KINDS = {"single": 0, "cluster7": 1, "ball": 2}

EXPORTS = ("ca_version", "ca_last_error", "ca_workspace_bytes", "ca_create", "ca_destroy", "ca_seed", "ca_set_rng",
           "ca_set_protocols", "ca_run", "ca_step", "ca_get_step", "ca_sync", "ca_fitness", "ca_counts",
           "ca_get_state", "ca_set_state", "ca_stage", "ca_set_option", "ca_get_option", "ca_launch_count",
           "ca_counts_noalloc")


class CaParams(C.Structure):
    """struct ca_params of include/ca.h"""
    _fields_ = [
        ("steps_per_hour", C.c_int32), ("n_sub", C.c_int32),
        ("lambda_", C.c_float * 3), ("boundary", C.c_float * 3),
        ("rate", (C.c_float * 4) * 3),
        ("O_A", C.c_float), ("G_P", C.c_float), ("G_Q", C.c_float), ("H_P", C.c_float), ("H_Q", C.c_float),
        ("T", C.c_int32 * 4), ("J", C.c_int32 * 4),
        ("alpha", C.c_float * 4), ("beta", C.c_float * 4),
        ("oer_m", C.c_float), ("oer_K", C.c_float),
        ("repair_period", C.c_int32), ("repair_shift", C.c_int32),
        ("lysis_steps", C.c_int32), ("N_ref", C.c_int32), ("well_mixed_medium", C.c_int32),
    ]


class CaInit(C.Structure):
    """struct ca_init of include/ca.h"""
    _fields_ = [("kind", C.c_int32), ("cx", C.c_int32), ("cy", C.c_int32), ("cz", C.c_int32),
                ("radius", C.c_float), ("shared_init", C.c_int32)]


class CaError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("libca_b200 error %d: %s" % (code, msg))
        self.code = code


_LIB = None


def load():
    """Load the in-tree CUDA library; raises (never falls back) if it is absent."""
    global _LIB
    if _LIB is not None:
        return _LIB
    if not os.path.exists(LIB_PATH):
        raise ImportError("%s is missing: run `python -m paper_2303_08123_b200.build` (there is no CPU fallback)" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.ca_version.restype = C.c_char_p
    L.ca_last_error.restype = C.c_char_p
    L.ca_last_error.argtypes = [vp]
    L.ca_workspace_bytes.restype = C.c_size_t
    L.ca_workspace_bytes.argtypes = [C.c_int] * 5
    L.ca_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int, C.c_int, C.POINTER(CaParams), C.c_int, vp, C.c_size_t, vp]
    L.ca_destroy.argtypes = [vp]
    L.ca_seed.argtypes = [vp, C.POINTER(CaInit), C.c_uint64, C.c_uint32]
    L.ca_set_rng.argtypes = [vp, C.c_uint64, C.c_uint32]
    L.ca_set_protocols.argtypes = [vp, vp, vp, vp, C.c_int, C.c_float]
    L.ca_run.argtypes = [vp, C.c_double]
    L.ca_step.argtypes = [vp, C.c_int64]
    L.ca_get_step.argtypes = [vp, C.POINTER(C.c_int64)]
    L.ca_sync.argtypes = [vp]
    L.ca_fitness.argtypes = [vp, vp, C.c_int]
    L.ca_counts.argtypes = [vp, vp, C.c_int]
    L.ca_get_state.argtypes = [vp, C.c_int, vp, vp, vp, vp, vp, vp, C.POINTER(C.c_int64)]
    L.ca_set_state.argtypes = [vp, C.c_int, C.c_int, vp, vp, vp, vp, vp, vp, C.c_int64]
    L.ca_stage.argtypes = [vp, C.c_int, C.c_int]
    L.ca_set_option.argtypes = [vp, C.c_char_p, C.c_int]
    L.ca_get_option.argtypes = [vp, C.c_char_p, C.POINTER(C.c_int)]
    L.ca_counts_noalloc.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, vp, vp, vp]
    L.ca_launch_count.argtypes = [vp]
    L.ca_launch_count.restype = C.c_int64
    _LIB = L
    return L


def make_params(d):
    """dict with the keys of workloads.default_params() -> CaParams"""
    p = CaParams()
    p.steps_per_hour = int(d["steps_per_hour"])
    p.n_sub = int(d["n_sub"])
    for s in range(3):
        p.lambda_[s] = d["lambda"][s]
        p.boundary[s] = d["boundary"][s]
        for m in range(4):
            p.rate[s][m] = d["rate"][s][m]
    for k in ("O_A", "G_P", "G_Q", "H_P", "H_Q", "oer_m", "oer_K"):
        setattr(p, k, d[k])
    for k in range(4):
        p.T[k] = int(d["T"][k])
        p.J[k] = int(d["J"][k])
        p.alpha[k] = d["alpha"][k]
        p.beta[k] = d["beta"][k]
    p.well_mixed_medium = int(d.get("well_mixed_medium", 0))
    for k in ("repair_period", "repair_shift", "lysis_steps", "N_ref"):
        setattr(p, k, int(d[k]))
    return p


def _ptr(a):
    return None if a is None else C.c_void_p(a.ctypes.data)


CA_NOALLOC_MAX_BATCH = 16384


def counts_noalloc(state, nx, ny, nz, n_ref=0, counts_out=None, fitness_out=None, stream=None):
    """ca_counts_noalloc: counts / Eq. 1 fitness of a torch cuda uint8 tensor `state` [batch][nz][ny][nx] into torch cuda tensors
    the caller passes (int32 [batch][CA_NCOUNT], fp32 [batch]); the library allocates nothing (fixed scratch, batch <= 16384)."""
    L = load()
    batch = int(state.shape[0])
    ptr = lambda t: None if t is None else C.c_void_p(t.data_ptr())
    rc = L.ca_counts_noalloc(ptr(state), batch, int(nx), int(ny), int(nz), int(n_ref), ptr(counts_out), ptr(fitness_out),
                             None if stream is None else C.c_void_p(stream.cuda_stream))
    if rc:
        raise CaError(rc, (L.ca_last_error(None) or b"").decode())


class CaBatch:
    """One ca_ctx: `batch` simulations on an nx*ny*nz lattice.  Methods mirror the C entry points
    (ca_seed -> seed, ca_set_protocols -> set_protocols, ca_run -> run, ca_fitness -> fitness, ...)."""

    def __init__(self, batch, nx, ny, nz, params, max_frac=10, device=0, stream=None):
        import torch
        self.L = load()
        if not torch.cuda.is_available():
            raise CaError(CA_ECUDA, "no CUDA device: libca_b200 has no CPU path")
        self.torch = torch
        self.device = torch.device("cuda", device)
        self.batch, self.nx, self.ny, self.nz = int(batch), int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.max_frac = int(max_frac)
        self.params = make_params(params)
        need = self.L.ca_workspace_bytes(self.batch, self.nx, self.ny, self.nz, self.max_frac)
        if need == 0:
            raise CaError(CA_EINVAL, "bad batch / lattice dims / max_frac")
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(need, dtype=torch.uint8, device=self.device)     # device memory from torch
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)   # stream from torch
            ctx = C.c_void_p()
            rc = self.L.ca_create(C.byref(ctx), self.batch, self.nx, self.ny, self.nz, C.byref(self.params), self.max_frac,
                                  C.c_void_p(self.workspace.data_ptr()), need, C.c_void_p(self.stream.cuda_stream))
        if rc:
            raise CaError(rc, (self.L.ca_last_error(None) or b"").decode())
        self.ctx = ctx

    def _chk(self, rc):
        if rc:
            raise CaError(rc, (self.L.ca_last_error(self.ctx) or b"").decode())

    def close(self):
        if getattr(self, "ctx", None):
            self.L.ca_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def seed(self, kind="cluster7", center=(-1, -1, -1), radius=0.0, shared_init=False, rng_seed=0, sim_id_base=0):
        init = CaInit(INIT_KINDS[kind], int(center[0]), int(center[1]), int(center[2]), float(radius), int(shared_init))
        self._chk(self.L.ca_seed(self.ctx, C.byref(init), int(rng_seed), int(sim_id_base)))

    def set_rng(self, rng_seed, sim_id_base=0):
        self._chk(self.L.ca_set_rng(self.ctx, int(rng_seed), int(sim_id_base)))

    def set_protocols(self, dose_gy, delay_h, nfrac=None, t0_h=0.0):
        d = np.ascontiguousarray(dose_gy, dtype=np.float32)
        t = np.ascontiguousarray(delay_h, dtype=np.float32)
        if d.ndim == 1:
            d, t = d[None, :], t[None, :]
        assert d.shape == t.shape and d.shape[0] == self.batch, (d.shape, t.shape, self.batch)
        nf = np.full(self.batch, d.shape[1], np.int32) if nfrac is None else np.ascontiguousarray(nfrac, dtype=np.int32)
        self._chk(self.L.ca_set_protocols(self.ctx, _ptr(d), _ptr(t), _ptr(nf), int(d.shape[1]), float(t0_h)))

    def run(self, t_end_h):
        self._chk(self.L.ca_run(self.ctx, float(t_end_h)))

    def step(self, n=1):
        self._chk(self.L.ca_step(self.ctx, int(n)))

    @property
    def step_index(self):
        s = C.c_int64()
        self._chk(self.L.ca_get_step(self.ctx, C.byref(s)))
        return int(s.value)

    def sync(self):
        self._chk(self.L.ca_sync(self.ctx))

    def fitness(self, out=None):
        """-> numpy [batch] fp32 (host), or fills a torch cuda tensor `out` asynchronously"""
        if out is not None:
            self._chk(self.L.ca_fitness(self.ctx, C.c_void_p(out.data_ptr()), 1))
            return out
        res = np.zeros(self.batch, np.float32)
        self._chk(self.L.ca_fitness(self.ctx, _ptr(res), 0))
        return res

    def counts(self):
        res = np.zeros((self.batch, CA_NCOUNT), np.int32)
        self._chk(self.L.ca_counts(self.ctx, _ptr(res), 0))
        return res

    def get_state(self, sim=0, fields=True):
        st = np.zeros(self.shape, np.uint8)
        ck = np.zeros(self.shape, np.uint16)
        dm = np.zeros(self.shape, np.uint16)
        f = [np.zeros(self.shape, np.float32) for _ in range(3)] if fields else [None] * 3
        s = C.c_int64()
        self._chk(self.L.ca_get_state(self.ctx, int(sim), _ptr(st), _ptr(ck), _ptr(dm), _ptr(f[0]), _ptr(f[1]), _ptr(f[2]), C.byref(s)))
        return dict(state=st, clock=ck, damage=dm, o2=f[0], glc=f[1], h=f[2], step=int(s.value))

    def set_state(self, sim_first=0, sim_count=None, state=None, clock=None, damage=None, o2=None, glc=None, h=None, step=-1):
        def prep(a, dt):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=dt)
            assert a.shape == self.shape, (a.shape, self.shape)
            return a
        n = self.batch - sim_first if sim_count is None else sim_count
        arrs = [prep(state, np.uint8), prep(clock, np.uint16), prep(damage, np.uint16),
                prep(o2, np.float32), prep(glc, np.float32), prep(h, np.float32)]
        self._chk(self.L.ca_set_state(self.ctx, int(sim_first), int(n), *[_ptr(a) for a in arrs], int(step)))

    def stage(self, stage, arg=0):
        self._chk(self.L.ca_stage(self.ctx, int(stage), int(arg)))

    def set_option(self, name, value):
        self._chk(self.L.ca_set_option(self.ctx, name.encode(), int(value)))

    def get_option(self, name):
        v = C.c_int()
        self._chk(self.L.ca_get_option(self.ctx, name.encode(), C.byref(v)))
        return int(v.value)

    @property
    def launch_count(self):
        return int(self.L.ca_launch_count(self.ctx))
