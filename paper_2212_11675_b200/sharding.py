"""Host logic of the multi-GPU row sharding (Fig. 2).

The paper splits the observation rows into contiguous, star-aligned blocks, one per process
(its N[nproc]).  The astrometric part of A is block diagonal by star
(PAPER.md:73), so the astrometric slice of every n-vector is DISTRIBUTED with its rows; the
attitude + instrumental + global slice is REPLICATED and summed over the processes after
every aprod2.  This module only computes the partition and the index maps;
it holds no arithmetic of the method and is shared by the product and by the CPU gloo test.

A shard is itself an ordinary system (gsr_matrix_create with S_local stars and the same D, I):
    local column j < 5*S_local           <-> global column 5*star0 + j
    local column 5*S_local + r           <-> global column 5*S + r     (replicated slice)
"""
from __future__ import annotations

from dataclasses import dataclass
from typing import List, Sequence


@dataclass(frozen=True)
class Shard:
    rank: int
    world: int
    star0: int      # first star of the block
    star1: int      # one past the last star
    row0: int       # first row
    row1: int       # one past the last row
    n_stars: int    # S of the whole system
    n_dfa: int
    n_instr: int

    @property
    def n_rows_local(self) -> int:
        return self.row1 - self.row0

    @property
    def n_stars_local(self) -> int:
        return self.star1 - self.star0

    @property
    def n_cols_local(self) -> int:
        return 5 * self.n_stars_local + self.n_replicated

    @property
    def n_replicated(self) -> int:
        """Length of the replicated slice: 3 D attitude + I instrumental + 1 global."""
        return 3 * self.n_dfa + self.n_instr + 1

    @property
    def replicated_offset_local(self) -> int:
        return 5 * self.n_stars_local

    @property
    def replicated_offset_global(self) -> int:
        return 5 * self.n_stars

    @property
    def astro_offset_global(self) -> int:
        return 5 * self.star0


def shard_rows(star_ptr: Sequence[int], world: int, n_dfa: int, n_instr: int) -> List[Shard]:
    """Contiguous star-aligned row blocks balanced by row count.

    star_ptr[s] is the first row of star s (length S+1, non-decreasing).  Block r ends at the
    star boundary closest to (r+1)*m/world; blocks may be empty when world > S."""
    S = len(star_ptr) - 1
    m = int(star_ptr[S])
    assert world >= 1 and S >= 1
    cuts = [0]
    s = 0
    for r in range(1, world):
        target = r * m / world
        while s < S and int(star_ptr[s + 1]) <= target:
            s += 1
        # s is the last boundary at or below the target; take s+1 if it is closer
        if s < S and (int(star_ptr[s + 1]) - target) < (target - int(star_ptr[s])):
            s += 1
        s = max(s, cuts[-1])
        cuts.append(s)
    cuts.append(S)
    return [Shard(r, world, cuts[r], cuts[r + 1], int(star_ptr[cuts[r]]), int(star_ptr[cuts[r + 1]]),
                  S, int(n_dfa), int(n_instr)) for r in range(world)]


def local_star_idx(star_idx, shard: Shard):
    """Star indices of the shard's rows, rebased to the shard (works on numpy / torch arrays)."""
    return star_idx[shard.row0:shard.row1] - shard.star0


def scatter_x(x_global, shard: Shard):
    """Local n-vector of a shard from a global one (astrometric slice + replicated slice)."""
    a0, r0 = shard.astro_offset_global, shard.replicated_offset_global
    import numpy as np
    return np.concatenate([x_global[a0:a0 + 5 * shard.n_stars_local], x_global[r0:]])


def gather_x(x_locals, shards: Sequence[Shard]):
    """Global n-vector from the shards' local ones (replicated slice taken from rank 0)."""
    import numpy as np
    astro = [x[:5 * sh.n_stars_local] for x, sh in zip(x_locals, shards)]
    return np.concatenate(astro + [x_locals[0][shards[0].replicated_offset_local:]])
