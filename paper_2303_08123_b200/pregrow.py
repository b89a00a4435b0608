"""Pre-grown tumours (tumours are grown once, saved, and re-loaded for every evaluation).

BASELINE configs[2] starts every simulation from one spheroid "grown from a single cell to ~1 mm diameter before
treatment": 64 sites across on the 96^3 lattice (G19).  The growth runs in libca_b200 on the GPU (one
simulation, no protocol); the snapshot is what `CaBatch.set_state` broadcasts to the batch.  Host code only."""
import numpy as np

from . import binding


def extent(state):
    """largest bounding-box side (in sites) of the occupied set of a (nz, ny, nx) state array; 0 if empty"""
    k = state & 7
    occ = (k >= 1) & (k <= 5)
    if not occ.any():
        return 0
    out = 0
    for ax in range(3):
        other = tuple(a for a in range(3) if a != ax)
        line = np.flatnonzero(occ.any(axis=other))
        out = max(out, int(line[-1] - line[0] + 1))
    return out


def grow(dims, params, init, rng_seed, target_extent=None, target_cells=None, check_h=12.0, max_h=4000.0, device=0, sim_id=0):
    """Grow ONE untreated simulation from `init` until its occupied set is `target_extent` sites across (or holds
    `target_cells` live cells).  Returns (snapshot dict as CaBatch.get_state gives it, hours grown)."""
    nx, ny, nz = dims
    g = binding.CaBatch(1, nx, ny, nz, params, max_frac=1, device=device)
    try:
        g.seed(rng_seed=rng_seed, sim_id_base=sim_id, **init)
        t = 0.0
        while t < max_h:
            t += check_h
            g.run(t)
            if target_cells is not None:
                if int(g.counts()[0, 0]) >= target_cells:
                    break
            elif extent(g.get_state(0, fields=False)["state"]) >= target_extent:
                break
        else:
            raise RuntimeError("tumour did not reach the target within %g h" % max_h)
        return g.get_state(0), t
    finally:
        g.close()


def radial_profile(snapshot, center=None):
    """mean radius (sites, from the centre of mass of the occupied set) of proliferating, quiescent and dead cells, and
    their counts: the rim / quiescent shell / necrotic core order of a spheroid."""
    st = snapshot["state"]
    k = st & 7
    live = (k >= 1) & (k <= 4)
    mode = (st >> 3) & 3
    z, y, x = np.indices(st.shape)
    occ = live | (k == 5)
    c = center if center is not None else (x[occ].mean(), y[occ].mean(), z[occ].mean())
    r = np.sqrt((x - c[0]) ** 2 + (y - c[1]) ** 2 + (z - c[2]) ** 2)
    sel = {"proliferating": live & (mode < 2), "quiescent": live & (mode >= 2), "dead": k == 5,
           "anaerobic": live & ((mode & 1) == 1)}
    out = {name: (int(m.sum()), float(r[m].mean()) if m.any() else float("nan")) for name, m in sel.items()}
    out["r_max"] = float(r[occ].max()) if occ.any() else 0.0
    # hollow core: EMPTY sites well inside the occupied ball (lysed necrotic cells)
    out["empty_inside_half_radius"] = int(((k == 0) & (r < 0.5 * out["r_max"])).sum())
    return out


def grow_library(dims, params, init, rng_seed, n_tumours, grow_h, device=0):
    """The tumour library of PAPER.md l.244: `n_tumours` untreated simulations from the same seed geometry, different
    simulation ids (0 .. n-1), grown for `grow_h` hours in ONE batch.  Returns the list of snapshots."""
    nx, ny, nz = dims
    g = binding.CaBatch(n_tumours, nx, ny, nz, params, max_frac=1, device=device)
    try:
        g.seed(rng_seed=rng_seed, sim_id_base=0, **init)
        g.run(grow_h)
        return [g.get_state(j) for j in range(n_tumours)]
    finally:
        g.close()
