"""Rank-grid arithmetic of the domain decomposition (host logic only: no arithmetic of the operator, no torch).

The global lattice L of extents (T, Z, Y, X) is cut into a grid of hyper-rectangular local lattices P_i
(eqs. 2.1-2.4), one per rank.  Rank order: the process coordinates (p_T, p_Z, p_Y, p_X) are numbered
like lattice sites, X fastest: rank = ((p_T * g_Z + p_Z) * g_Y + p_Y) * g_X + p_X.  The seams are periodic:
the neighbour of the last sub-lattice in a direction is the first one.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


def default_grid(world_size: int, global_dims) -> tuple:
    """Split T first (up to 4 ways), then Z, then Y, then X — powers of two, local extents kept >= 4 and even."""
    grid = [1, 1, 1, 1]
    n = world_size
    while n > 1:
        if n % 2:
            raise ValueError("world size must be a power of two")
        for mu in range(4):
            local = global_dims[mu] // grid[mu]
            if grid[mu] < 4 and local % 2 == 0 and local // 2 >= 4:
                grid[mu] *= 2
                break
        else:
            raise ValueError("lattice too small for this many ranks")
        n //= 2
    return tuple(grid)


@dataclass(frozen=True)
class Decomposition:
    global_dims: tuple
    grid: tuple

    def __post_init__(self):
        for n, g in zip(self.global_dims, self.grid):
            if g < 1 or n % g:
                raise ValueError("the process grid must divide the global lattice")

    @property
    def world_size(self) -> int:
        return int(np.prod(self.grid))

    @property
    def local_dims(self) -> tuple:
        return tuple(n // g for n, g in zip(self.global_dims, self.grid))

    @property
    def decomposed(self) -> tuple:
        return tuple(mu for mu in range(4) if self.grid[mu] > 1)

    def coords(self, rank: int) -> tuple:
        c = []
        for g in reversed(self.grid):
            c.append(rank % g)
            rank //= g
        return tuple(reversed(c))

    def rank(self, coords) -> int:
        r = 0
        for c, g in zip(coords, self.grid):
            r = r * g + (c % g)
        return r

    def neighbour(self, rank: int, mu: int, sign: int) -> int:
        """Rank that holds the sub-lattice next to `rank` in direction +mu (sign = +1) or -mu (sign = -1)."""
        c = list(self.coords(rank))
        c[mu] += sign
        return self.rank(c)

    def origin(self, rank: int) -> tuple:
        return tuple(c * n for c, n in zip(self.coords(rank), self.local_dims))

    def local_slices(self, rank: int, halo: int = 0) -> tuple:
        """Index arrays (one per direction) of the global coordinates of the local lattice, optionally extended by
        `halo` sites on both sides of every DECOMPOSED direction (periodic wrap of the global lattice)."""
        out = []
        for mu in range(4):
            o, n, N = self.origin(rank)[mu], self.local_dims[mu], self.global_dims[mu]
            h = halo if self.grid[mu] > 1 else 0
            out.append(np.arange(o - h, o + n + h) % N)
        return tuple(out)

    def extract(self, field: np.ndarray, rank: int, halo: int = 0) -> np.ndarray:
        """Local part of a canonical site-major global field [V_global, ...] -> [V_local(+halo), ...] (a copy)."""
        T, Z, Y, X = self.global_dims
        f = field.reshape(T, Z, Y, X, *field.shape[1:])
        t, z, y, x = self.local_slices(rank, halo)
        sub = f[np.ix_(t, z, y, x)]
        return np.ascontiguousarray(sub.reshape(-1, *field.shape[1:]))

    def insert(self, field: np.ndarray, rank: int, local: np.ndarray) -> None:
        """Write a local canonical field back into the global one."""
        T, Z, Y, X = self.global_dims
        f = field.reshape(T, Z, Y, X, *field.shape[1:])
        t, z, y, x = self.local_slices(rank)
        f[np.ix_(t, z, y, x)] = local.reshape(len(t), len(z), len(y), len(x), *field.shape[1:])

    def global_sites(self, rank: int, halo: int = 0) -> np.ndarray:
        """Canonical global site index of every site of the (extended) local lattice, in local canonical order."""
        T, Z, Y, X = self.global_dims
        t, z, y, x = self.local_slices(rank, halo)
        g = ((t[:, None, None, None] * Z + z[None, :, None, None]) * Y + y[None, None, :, None]) * X + x[None, None, None, :]
        return np.ascontiguousarray(g.reshape(-1)).astype(np.int64)

    def face_global_sites(self, rank: int, mu: int, high: bool) -> np.ndarray:
        """Global site index of the sites of the low / high face of direction mu, in face order (canonical order of
        the three remaining coordinates, X fastest — the order of the buffers of wd_dd_pack / wd_dd_exterior)."""
        T, Z, Y, X = self.global_dims
        sl = list(self.local_slices(rank))
        sl[mu] = sl[mu][-1:] if high else sl[mu][:1]
        t, z, y, x = sl
        g = ((t[:, None, None, None] * Z + z[None, :, None, None]) * Y + y[None, None, :, None]) * X + x[None, None, None, :]
        return np.ascontiguousarray(g.reshape(-1)).astype(np.int64)

    def interior_of_extended(self, halo: int) -> np.ndarray:
        """Positions, inside a local lattice extended by `halo`, of the sites of the local lattice itself."""
        ext = [n + (2 * halo if g > 1 else 0) for n, g in zip(self.local_dims, self.grid)]
        idx = np.arange(int(np.prod(ext))).reshape(ext)
        sl = tuple(slice(halo, halo + n) if g > 1 else slice(0, n) for n, g in zip(self.local_dims, self.grid))
        return np.ascontiguousarray(idx[sl].reshape(-1))

    def extended_dims(self, halo: int) -> tuple:
        return tuple(n + (2 * halo if g > 1 else 0) for n, g in zip(self.local_dims, self.grid))
