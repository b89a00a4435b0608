"""Shared test helpers: lattice construction only (no method arithmetic)."""
import numpy as np

K_EMPTY, K_G1, K_S, K_G2, K_M, K_DEAD, K_WALL = 0, 1, 2, 3, 4, 5, 7
ST_READY, ST_DOOMED = 0x20, 0x40


def blank_state(nx, ny, nz):
    """u8 lattice (nz, ny, nx): WALL on the outer layer, EMPTY inside (reading G2)."""
    st = np.full((nz, ny, nx), K_WALL, np.uint8)
    st[1:-1, 1:-1, 1:-1] = K_EMPTY
    return st


def const_fields(params, shape, dtype=np.float64):
    b = np.asarray(params["boundary"], dtype=np.float32).astype(dtype)
    return [np.full(shape, b[s], dtype) for s in range(3)]


def kind(st):
    return st & 7


def live(st):
    k = st & 7
    return (k >= 1) & (k <= 4)


def rel_err(a, b, floor):
    """|a-b| / max(|b|, floor), computed in fp64 (SURVEY.md 8(c) comparison protocol)."""
    a = np.asarray(a, np.float64)
    b = np.asarray(b, np.float64)
    return np.abs(a - b) / np.maximum(np.abs(b), floor)
