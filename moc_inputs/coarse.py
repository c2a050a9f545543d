"""Coarse (CMFD) meshes for the seeded test problems: a Cartesian overlay of the bounding rectangle.

Holds geometry only -- which coarse cell a triangle belongs to and the area / centre-distance ratio of a coarse
surface -- and none of the method's arithmetic; used by the oracle's tests and by the GPU parity tests alike.
"""
import numpy as np


def cartesian_cells(mesh, nx: int, ny: int) -> np.ndarray:
    """cell[r] = iy * nx + ix of the overlay cell that holds the centroid of triangle r."""
    c = mesh.xy[mesh.tri].mean(axis=1)
    ix = np.minimum((c[:, 0] / mesh.W * nx).astype(np.int64), nx - 1)
    iy = np.minimum((c[:, 1] / mesh.H * ny).astype(np.int64), ny - 1)
    return (iy * nx + ix).astype(np.int32)


def cartesian_coupling(mesh, nx: int, ny: int):
    """Returns f(lo, hi) -> A_s / d_s of the surface between overlay cells lo and hi (per unit height): hy / hx for
    x-neighbours, hx / hy for y-neighbours, 0 for any other pair (cells that only touch through the ragged edge of
    centroid-assigned triangles)."""
    hx, hy = mesh.W / nx, mesh.H / ny

    def f(lo, hi):
        lo, hi = np.asarray(lo, np.int64), np.asarray(hi, np.int64)
        dx, dy = np.abs(hi % nx - lo % nx), np.abs(hi // nx - lo // nx)
        return np.where((dx == 1) & (dy == 0), hy / hx, np.where((dx == 0) & (dy == 1), hx / hy, 0.0))
    return f
