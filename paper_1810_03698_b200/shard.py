"""Target sharding across GPUs: the host-side description of the exchange layout.

The arithmetic of the sharded matvec runs in the CUDA library (include/pb.h: pb_set_shard); this module states, in
numpy, the two index maps its kernels implement, so that the world_size-2 gloo test can exercise the exchange without
a GPU and the GPU test can check the kernels against it:

  pack_owned      = what k_combine writes into the all-gather send buffer: the owned rows of y in MORTON order,
                    [2][nmax] (row 1 of Eq. (5), then row 2), zero padded to the largest owned count nmax;
  unpack_gathered = what k_shard_scatter does after the all-gather: rank r's block [2][nmax] holds the Morton panels
                    first[r] .. first[r + 1]; panel i goes to y[perm[i]] and y[N + perm[i]] (original panel order).

No method arithmetic here (no kernels, quadrature or operators)."""
from __future__ import annotations

import numpy as np


def group_ranges_to_panels(first_group, n_panels: int, group_size: int = 64):
    """Group boundaries [world + 1] (pb_shard_partition) -> Morton panel boundaries."""
    return np.minimum(np.asarray(first_group, dtype=np.int64) * group_size, n_panels)


def nmax_of(first) -> int:
    first = np.asarray(first, dtype=np.int64)
    return int(np.max(first[1:] - first[:-1])) if first.size > 1 else 0


def pack_owned(y_morton, first, rank: int):
    """y_morton [2][N] (both rows of Eq. (5) in Morton order) -> this rank's send buffer, flat [2 * nmax]."""
    y_morton = np.asarray(y_morton, dtype=np.float64)
    nmax = nmax_of(first)
    i0, i1 = int(first[rank]), int(first[rank + 1])
    out = np.zeros((2, nmax))
    out[:, : i1 - i0] = y_morton[:, i0:i1]
    return out.reshape(-1)


def unpack_gathered(yall, first, perm):
    """yall flat [world * 2 * nmax] (the gathered send buffers, rank-major) -> y [2 N] in the original panel order."""
    first = np.asarray(first, dtype=np.int64)
    perm = np.asarray(perm, dtype=np.int64)
    world, nmax, N = first.size - 1, nmax_of(first), perm.size
    blocks = np.asarray(yall, dtype=np.float64).reshape(world, 2, nmax)
    y = np.empty(2 * N)
    for r in range(world):
        i0, i1 = int(first[r]), int(first[r + 1])
        y[perm[i0:i1]] = blocks[r, 0, : i1 - i0]
        y[N + perm[i0:i1]] = blocks[r, 1, : i1 - i0]
    return y
