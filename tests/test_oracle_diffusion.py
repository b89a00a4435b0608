"""Pins P3-P6: the oracle's reaction-diffusion stage O-S1 against a closed
form, a dense direct solve, and two invariants.  None of these re-use the oracle's own formula."""
import numpy as np
import pytest

from oracle import ca_oracle as o
from paper_2303_08123_b200 import workloads as w
from tests._helpers import blank_state, const_fields, K_G1


def _mode(shape):
    nz, ny, nx = shape
    z = np.sin(np.pi * np.arange(nz) / (nz - 1))
    y = np.sin(np.pi * np.arange(ny) / (ny - 1))
    x = np.sin(np.pi * np.arange(nx) / (nx - 1))
    m = z[:, None, None] * y[None, :, None] * x[None, None, :]
    m[0], m[-1], m[:, 0], m[:, -1], m[:, :, 0], m[:, :, -1] = 0, 0, 0, 0, 0, 0   # exactly zero on WALL
    return m


@pytest.mark.parametrize("dims", [(32, 32, 32), (20, 14, 9)])
def test_p3_mode_decay_closed_form(dims):
    """No cells; c = c_b + A*mode decays by g = 1 - 2*lam*sum_dim(1 - cos(pi/(n_dim-1))) per sub-step,
    exactly, for the discrete 7-point operator on an all-Dirichlet box."""
    nx, ny, nz = dims
    p = w.default_params()
    sim = o.OracleSim(nx, ny, nz, p)
    shape = (nz, ny, nx)
    b = np.asarray(p["boundary"], np.float32).astype(np.float64)
    lam = np.asarray(p["lambda"], np.float32).astype(np.float64)
    A = 0.25 * b
    mode = _mode(shape)
    f = [b[s] + A[s] * mode for s in range(3)]
    sim.set_state(state=blank_state(nx, ny, nz), clock=np.zeros(shape, np.uint16), damage=np.zeros(shape, np.uint16),
                  o2=f[0], glc=f[1], h=f[2], step=0)
    m = 1000
    sim.diffuse_substeps(m)
    out = sim.get_state()
    geo = sum(1.0 - np.cos(np.pi / (n - 1)) for n in dims)
    for s, name in enumerate(("o2", "glc", "h")):
        g = 1.0 - 2.0 * lam[s] * geo
        expect = b[s] + A[s] * g ** m * mode
        err = np.abs(out[name] - expect).max() / A[s]
        assert err < 1e-12, (name, err)
    if dims == (32, 32, 32):      # the number SURVEY.md 8(c) P3 prints for n = 32, lambda = 0.15
        assert abs((1.0 - 2.0 * lam[0] * geo) - 0.995382391) < 2e-8   # lam is fp32(0.15)


def test_p3_mode_decay_fp32_diagnostic_build():
    nx = ny = nz = 32
    p = w.default_params()
    sim = o.OracleSim(nx, ny, nz, p, precision="f32")
    shape = (nz, ny, nx)
    b = np.asarray(p["boundary"], np.float32).astype(np.float64)
    lam = np.asarray(p["lambda"], np.float32).astype(np.float64)
    mode = _mode(shape)
    f = [b[s] + 0.25 * b[s] * mode for s in range(3)]
    sim.set_state(state=blank_state(nx, ny, nz), o2=f[0], glc=f[1], h=f[2], step=0)
    sim.diffuse_substeps(1000)
    out = sim.get_state()
    geo = 3 * (1.0 - np.cos(np.pi / 31))
    for s, name in enumerate(("o2", "glc", "h")):
        expect = b[s] + 0.25 * b[s] * (1.0 - 2.0 * lam[s] * geo) ** 1000 * mode
        assert (np.abs(out[name] - expect) / b[s]).max() < 1e-5


def test_p4_steady_state_matches_dense_direct_solve():
    """6^3 lattice (64 unknowns): frozen sinks, iterate O-S1 to convergence, compare with
    numpy.linalg.solve of  lam * L c = -r  with Dirichlet data moved to the right-hand side."""
    n = 6
    p = w.default_params()
    shape = (n, n, n)
    rng = np.random.default_rng(11)
    st = blank_state(n, n, n)
    # an arbitrary pattern of live cells in mode PA (mode bits 0): frozen because only diffuse runs
    occ = rng.random((n - 2, n - 2, n - 2)) < 0.4
    st[1:-1, 1:-1, 1:-1][occ] = K_G1
    sim = o.OracleSim(n, n, n, p)
    f = const_fields(p, shape)
    sim.set_state(state=st, clock=np.zeros(shape, np.uint16), damage=np.zeros(shape, np.uint16),
                  o2=f[0], glc=f[1], h=f[2], step=0)
    sim.diffuse_substeps(4000)
    out = sim.get_state()
    idx = -np.ones(shape, int)
    interior = [(z, y, x) for z in range(1, n - 1) for y in range(1, n - 1) for x in range(1, n - 1)]
    for k, q in enumerate(interior):
        idx[q] = k
    for s, name in enumerate(("o2", "glc", "h")):
        lam = float(np.float32(p["lambda"][s]))
        cb = float(np.float32(p["boundary"][s]))
        r = float(np.float32(p["rate"][s][0]))
        Amat = np.zeros((len(interior), len(interior)))
        rhs = np.zeros(len(interior))
        for k, (z, y, x) in enumerate(interior):
            Amat[k, k] = -6.0 * lam
            rhs[k] = -(r if occ[z - 1, y - 1, x - 1] else 0.0)
            for dz, dy, dx in ((0, 0, 1), (0, 0, -1), (0, 1, 0), (0, -1, 0), (1, 0, 0), (-1, 0, 0)):
                j = idx[z + dz, y + dy, x + dx]
                if j >= 0:
                    Amat[k, j] = lam
                else:
                    rhs[k] -= lam * cb
        sol = np.linalg.solve(Amat, rhs)
        got = np.array([out[name][q] for q in interior])
        assert np.abs(got - sol).max() / cb < 1e-10, name
        assert (out[name][st == 7] == cb).all()


def test_p4_radial_profile_of_a_ball_of_sinks():
    """32^3, BALL of fixed sinks: field monotone in r, centre deficit within 15 % of q R^2/(2 lam)... the
    continuum estimate (ball term q R^2/6lam + exterior term ~ q R^2/3lam) ignores the finite box, which
    LOWERS the deficit; accept 0.6..1.15 of the estimate and require monotonicity along an axis."""
    n, R = 32, 6
    p = w.default_params()
    shape = (n, n, n)
    st = blank_state(n, n, n)
    zz, yy, xx = np.meshgrid(np.arange(n), np.arange(n), np.arange(n), indexing="ij")
    r2 = (zz - 16) ** 2 + (yy - 16) ** 2 + (xx - 16) ** 2
    st[r2 <= R * R] = K_G1            # mode PA
    sim = o.OracleSim(n, n, n, p)
    f = const_fields(p, shape)
    sim.set_state(state=st, o2=f[0], glc=f[1], h=f[2], step=0)
    sim.diffuse_substeps(6000)
    o2 = sim.get_state()["o2"]
    q = -float(np.float32(p["rate"][0][0]))
    lam = float(np.float32(p["lambda"][0]))
    cb = float(np.float32(p["boundary"][0]))
    deficit = cb - o2[16, 16, 16]
    est = q * R * R / (2 * lam)
    assert 0.6 * est < deficit < 1.15 * est, (deficit, est)
    line = o2[16, 16, 16:]
    assert (np.diff(line) > 0).all()          # strictly increasing from the centre to the wall


def test_p5_uniform_field_is_reproduced_bit_exactly():
    for precision in ("f64", "f32"):
        p = w.default_params()
        sim = o.OracleSim(16, 12, 10, p, precision=precision)
        sim.seed("single", rng_seed=1)
        st = sim.get_state()
        sim.set_state(state=blank_state(16, 12, 10), clock=np.zeros_like(st["clock"]))   # remove the cell
        before = sim.get_state()
        sim.step(300)
        after = sim.get_state()
        for name in ("o2", "glc", "h"):
            assert np.array_equal(before[name], after[name]), (precision, name)
            assert np.unique(after[name]).size == 1


def test_p6_mass_balance_and_maximum_principle():
    """sum_interior(c' - c) = lam * sum_{faces to WALL}(c_wall - c_site) + sum r  (interior-interior fluxes
    cancel pairwise), while no clamp fires; O2/glucose never exceed, H+ never undercuts, the boundary."""
    n = 14
    p = w.default_params()
    shape = (n, n, n)
    rng = np.random.default_rng(5)
    st = blank_state(n, n, n)
    occ = rng.random((n - 2,) * 3) < 0.3
    modes = rng.integers(0, 4, (n - 2,) * 3).astype(np.uint8)
    inner = st[1:-1, 1:-1, 1:-1]
    inner[occ] = (K_G1 | (modes[occ] << 3))
    sim = o.OracleSim(n, n, n, p)
    f = const_fields(p, shape)
    sim.set_state(state=st, o2=f[0], glc=f[1], h=f[2], step=0)
    for it in range(40):
        a = sim.get_state()
        sim.diffuse_substeps(1)
        b = sim.get_state()
        for s, name in enumerate(("o2", "glc", "h")):
            lam = float(np.float32(p["lambda"][s]))
            cb = float(np.float32(p["boundary"][s]))
            c = a[name]
            ci = c[1:-1, 1:-1, 1:-1]
            wall_flux = 0.0
            for ax in range(3):
                lo = np.take(ci, 0, axis=ax)
                hi = np.take(ci, -1, axis=ax)
                wall_flux += (cb - lo).sum() + (cb - hi).sum()
            rates = np.asarray(p["rate"][s], np.float32).astype(np.float64)
            src = rates[modes[occ]].sum()
            lhs = (b[name][1:-1, 1:-1, 1:-1] - ci).sum()
            rhs = lam * wall_flux + src
            scale = abs(src) + lam * abs(wall_flux) + 1e-300
            assert abs(lhs - rhs) / scale < 1e-9, (it, name, lhs, rhs)
            if s < 2:
                assert b[name].max() <= cb
            else:
                assert b[name].min() >= cb
            assert b[name].min() > 0.0          # no clamp fired


def test_well_mixed_medium_closed_forms_and_pinned_empty_sites():
    """Alternative reading of G2 ("well-mixed replenished substrate"; the `well_mixed_medium` flag of
    NEXT-3): every EMPTY site is held at the medium value.  Closed forms that do not re-use the oracle's formula:
    an isolated consuming cell sees six medium neighbours, so its fixed point is c* = c_b + r / (6 lambda);
    two face-adjacent identical cells see five medium neighbours and each other: c* = c_b + r / (5 lambda).
    EMPTY sites stay at the boundary value bit for bit; without the flag they do not."""
    n = 9
    p = w.default_params(well_mixed_medium=1)
    b = np.asarray(p["boundary"], np.float32).astype(np.float64)
    lam = np.asarray(p["lambda"], np.float32).astype(np.float64)
    rate = np.asarray(p["rate"], np.float32).astype(np.float64)
    shape = (n, n, n)
    for cells, nb in (([(4, 4, 4)], 6.0), ([(4, 4, 4), (4, 4, 5)], 5.0)):
        st = blank_state(n, n, n)
        for c in cells:
            st[c] = K_G1                                      # mode bits 0 = PA
        f = const_fields(p, shape)
        sim = o.OracleSim(n, n, n, p)
        sim.set_state(state=st, clock=np.full(shape, 1000, np.uint16), damage=np.zeros(shape, np.uint16), o2=f[0], glc=f[1], h=f[2], step=0)
        sim.diffuse_substeps(400)
        out = sim.get_state()
        for s, name in enumerate(("o2", "glc", "h")):
            expect = b[s] + rate[s][0] / (nb * lam[s])
            for c in cells:
                assert abs(out[name][c] - expect) <= 1e-12 * abs(expect), (name, c, out[name][c], expect)
            empty = (st == 0)
            assert np.array_equal(out[name][empty], np.full(empty.sum(), b[s]))       # pinned, bitwise
    # the same isolated cell WITHOUT the flag: its neighbours are depleted (free diffusion), the centre lies lower
    p0 = w.default_params()
    st = blank_state(n, n, n); st[4, 4, 4] = K_G1
    f = const_fields(p0, shape)
    sim = o.OracleSim(n, n, n, p0)
    sim.set_state(state=st, clock=np.full(shape, 1000, np.uint16), damage=np.zeros(shape, np.uint16), o2=f[0], glc=f[1], h=f[2], step=0)
    sim.diffuse_substeps(400)
    out = sim.get_state()
    assert out["glc"][4, 4, 5] < b[1] and out["glc"][4, 4, 4] < b[1] + rate[1][0] / (6.0 * lam[1])
