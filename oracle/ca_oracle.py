"""ORACLE binding (test infrastructure, NOT the product).

ctypes wrapper around oracle/ca_oracle.c -- the plain single-threaded CPU
simulator of the hot path (see ca_oracle.h for what it computes and which
passages of PAPER.md / readings of DESIGN.md it follows).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs may import this module.  It imports nothing from the
product package and the product package imports nothing from here.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "ca_oracle.c"), os.path.join(_HERE, "ca_oracle.h")]
C_NCOUNT = 13
COUNT_NAMES = ("live", "doomed", "ready", "dead", "G1", "S", "G2", "M", "PA", "PN", "QA", "QN", "occupied")


class CarParams(C.Structure):
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


class CarInit(C.Structure):
    _fields_ = [("kind", C.c_int32), ("cx", C.c_int32), ("cy", C.c_int32), ("cz", C.c_int32),
                ("radius", C.c_float), ("shared_init", C.c_int32)]


INIT_KINDS = {"single": 0, "cluster7": 1, "ball": 2}


def _lib_path(precision):
    return os.path.join(_HERE, "libca_oracle_%s.so" % precision)


def build(force=False):
    """Compile both precisions of the oracle with gcc (plain -O2, no contraction)."""
    for precision, defs in (("f64", []), ("f32", ["-DCA_REAL=float", "-DCA_REAL_IS_FLOAT"])):
        out = _lib_path(precision)
        if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(s) for s in _SRC):
            continue
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off", "-Wall", "-Wextra",
               *defs, "-o", out, _SRC[0], "-lm"]
        subprocess.check_call(cmd)


_LIBS = {}


def _lib(precision):
    if precision not in _LIBS:
        build()
        L = C.CDLL(_lib_path(precision))
        vp, u8p, u16p, dp, i64p, i32p = C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p
        L.car_create.restype = vp
        L.car_create.argtypes = [C.c_int, C.c_int, C.c_int, C.POINTER(CarParams)]
        L.car_destroy.argtypes = [vp]
        L.car_seed.argtypes = [vp, C.POINTER(CarInit), C.c_uint64, C.c_uint32]
        L.car_set_rng.argtypes = [vp, C.c_uint64, C.c_uint32]
        L.car_set_protocol.argtypes = [vp, dp, dp, C.c_int, C.c_double]
        L.car_fire_steps.argtypes = [vp, i64p, C.c_int]
        for name in ("car_stage_irradiate", "car_stage_diffuse", "car_stage_cells"):
            getattr(L, name).argtypes = [vp]
            getattr(L, name).restype = None
        L.car_stage_divide.argtypes = [vp]
        L.car_diffuse_substeps.argtypes = [vp, C.c_int]
        L.car_diffuse_substeps.restype = None
        L.car_step.argtypes = [vp, C.c_int64]
        L.car_step.restype = None
        L.car_run.argtypes = [vp, C.c_double]
        L.car_get_step.argtypes = [vp]
        L.car_get_step.restype = C.c_int64
        L.car_counts.argtypes = [vp, i32p]
        L.car_counts.restype = None
        L.car_fitness.argtypes = [vp]
        L.car_fitness.restype = C.c_double
        L.car_get_state.argtypes = [vp, u8p, u16p, u16p, dp, dp, dp]
        L.car_get_state.restype = None
        L.car_set_state.argtypes = [vp, u8p, u16p, u16p, dp, dp, dp, C.c_int64]
        L.car_philox4x32_10.argtypes = [C.POINTER(C.c_uint32 * 4), C.POINTER(C.c_uint32 * 2), C.POINTER(C.c_uint32 * 4)]
        L.car_philox4x32_10.restype = None
        L.car_uniform_int.argtypes = [C.c_uint32, C.c_uint32]
        L.car_uniform_int.restype = C.c_uint32
        L.car_bernoulli_threshold.argtypes = [C.c_double]
        L.car_bernoulli_threshold.restype = C.c_uint32
        L.car_real_bytes.restype = C.c_int
        _LIBS[precision] = L
    return _LIBS[precision]


def make_params(d):
    """dict (see paper_2303_08123_b200.workloads.default_params for the keys) -> CarParams."""
    p = CarParams()
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


def philox4x32_10(ctr, key, precision="f64"):
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    _lib(precision).car_philox4x32_10(C.byref(c), C.byref(k), C.byref(o))
    return [int(v) for v in o]


def uniform_int(x, m):
    return int(_lib("f64").car_uniform_int(int(x), int(m)))


def bernoulli_threshold(p):
    return int(_lib("f64").car_bernoulli_threshold(float(p)))


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleSim:
    """One simulation.  Arrays are numpy, shape (nz, ny, nx), x fastest."""

    def __init__(self, nx, ny, nz, params, precision="f64"):
        self.L = _lib(precision)
        self.precision = precision
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.shape = (self.nz, self.ny, self.nx)
        self.params = make_params(params)
        self.ctx = self.L.car_create(self.nx, self.ny, self.nz, C.byref(self.params))
        if not self.ctx:
            raise ValueError("car_create rejected the dimensions / parameters")

    def __del__(self):
        if getattr(self, "ctx", None):
            self.L.car_destroy(self.ctx)
            self.ctx = None

    def seed(self, kind="cluster7", center=(-1, -1, -1), radius=0.0, shared_init=False, rng_seed=0, sim_id=0):
        init = CarInit(INIT_KINDS[kind], int(center[0]), int(center[1]), int(center[2]), float(radius), int(shared_init))
        rc = self.L.car_seed(self.ctx, C.byref(init), int(rng_seed), int(sim_id))
        if rc:
            raise ValueError("car_seed failed")

    def set_rng(self, rng_seed, sim_id):
        self.L.car_set_rng(self.ctx, int(rng_seed), int(sim_id))

    def set_protocol(self, dose_gy, delay_h, t0_h=0.0):
        d = np.ascontiguousarray(dose_gy, dtype=np.float64)
        t = np.ascontiguousarray(delay_h, dtype=np.float64)
        assert d.shape == t.shape and d.ndim == 1
        rc = self.L.car_set_protocol(self.ctx, _ptr(d), _ptr(t), int(d.size), float(t0_h))
        if rc:
            raise ValueError("car_set_protocol rejected the protocol (rc=%d)" % rc)

    def fire_steps(self):
        out = np.zeros(64, dtype=np.int64)
        n = self.L.car_fire_steps(self.ctx, _ptr(out), 64)
        return out[:n].copy()

    def stage_irradiate(self):
        self.L.car_stage_irradiate(self.ctx)

    def stage_diffuse(self):
        self.L.car_stage_diffuse(self.ctx)

    def stage_cells(self):
        self.L.car_stage_cells(self.ctx)

    def stage_divide(self):
        return int(self.L.car_stage_divide(self.ctx))

    def diffuse_substeps(self, m):
        self.L.car_diffuse_substeps(self.ctx, int(m))

    def step(self, n=1):
        self.L.car_step(self.ctx, int(n))

    def run(self, t_end_h):
        rc = self.L.car_run(self.ctx, float(t_end_h))
        if rc:
            raise ValueError("car_run: t_end lies in the past")

    @property
    def step_index(self):
        return int(self.L.car_get_step(self.ctx))

    def counts(self):
        out = np.zeros(C_NCOUNT, dtype=np.int32)
        self.L.car_counts(self.ctx, _ptr(out))
        return out

    def fitness(self):
        return float(self.L.car_fitness(self.ctx))

    def get_state(self):
        """-> dict(state u8, clock u16, damage u16, o2/glc/h float64, step)"""
        st = np.zeros(self.shape, np.uint8)
        ck = np.zeros(self.shape, np.uint16)
        dm = np.zeros(self.shape, np.uint16)
        f = [np.zeros(self.shape, np.float64) for _ in range(3)]
        self.L.car_get_state(self.ctx, _ptr(st), _ptr(ck), _ptr(dm), _ptr(f[0]), _ptr(f[1]), _ptr(f[2]))
        return dict(state=st, clock=ck, damage=dm, o2=f[0], glc=f[1], h=f[2], step=self.step_index)

    def set_state(self, state=None, clock=None, damage=None, o2=None, glc=None, h=None, step=-1):
        def prep(a, dt):
            if a is None:
                return None
            a = np.ascontiguousarray(a, dtype=dt)
            assert a.shape == self.shape, (a.shape, self.shape)
            return a
        st, ck, dm = prep(state, np.uint8), prep(clock, np.uint16), prep(damage, np.uint16)
        f = [prep(o2, np.float64), prep(glc, np.float64), prep(h, np.float64)]
        self.L.car_set_state(self.ctx, _ptr(st), _ptr(ck), _ptr(dm), _ptr(f[0]), _ptr(f[1]), _ptr(f[2]), int(step))
