"""Host-side partition of the (partial wave, energy) units over ranks: one process per GPU.

Every (wave, energy) R-matrix of eq. 4 is independent, so the path shards with
no data-path collective: "the loop in energy is the one which is parallelised, the energy array
is split among the processors nproc, so each processor is assigned a set of nproce = NE/nproc
energies".  PSTGF v1.1 makes the energy set a rank works on depend on the partial
wave, "so the amount of fast energies and slow energies calculated by each processor is evenly
distributed ... all processors calculate all energies, but never consecutive energies for the
same partial wave" (Fig. 1 at :141), and starts every rank on a different
partial wave so that they do not all read the same H.DATXXX at once (:145).

Reading (R13): the mesh of a wave is cut into blocks of ``block`` consecutive
energies (the kernel's energy block, so that no block is split between GPUs); block b belongs
to energy set ``b mod world``; on wave p rank r works set ``(r + p) mod world``; rank r visits
the waves in the order ``r, r+1, ..., P-1, 0, ..., r-1`` (the oval of Fig. 1).  This module is
index arithmetic only: none of the method's arithmetic lives here.
"""
from __future__ import annotations

import numpy as np

ENERGY_BLOCK = 8   # energies per work item of the kernel (csrc/rmat_common.h: EB)


def energy_set_of_rank(wave_index: int, rank: int, world: int) -> int:
    """The energy set rank ``rank`` works on for wave ``wave_index`` (Fig. 1, right: v1.1)."""
    if not (0 <= rank < world):
        raise ValueError("rank must be in [0, world)")
    return (rank + wave_index) % world


def energy_indices(n_E: int, wave_index: int, rank: int, world: int, block: int = ENERGY_BLOCK) -> np.ndarray:
    """Indices (ascending) into a wave's mesh of the energies rank ``rank`` forms R for."""
    if n_E < 0 or world < 1 or block < 1:
        raise ValueError("n_E >= 0, world >= 1, block >= 1 required")
    s = energy_set_of_rank(wave_index, rank, world)
    n_blocks = -(-n_E // block)
    mine = np.arange(s, n_blocks, world, dtype=np.int64)
    idx = (mine[:, None] * block + np.arange(block, dtype=np.int64)[None, :]).ravel()
    return idx[idx < n_E]


def wave_order(n_waves: int, rank: int, world: int) -> list[int]:
    """The order in which rank ``rank`` visits the partial waves (each rank starts on another one)."""
    if n_waves == 0:
        return []
    start = rank % n_waves
    return [(start + i) % n_waves for i in range(n_waves)]


def plan(n_E_per_wave, rank: int, world: int, block: int = ENERGY_BLOCK) -> list[tuple[int, np.ndarray]]:
    """[(wave index, energy indices)] for this rank, in its visiting order.  Waves for which the
    rank has no energies are kept (with an empty index array) so that every rank sees every wave."""
    n_waves = len(n_E_per_wave)
    return [(p, energy_indices(int(n_E_per_wave[p]), p, rank, world, block)) for p in wave_order(n_waves, rank, world)]


def counts(n_E_per_wave, world: int, block: int = ENERGY_BLOCK) -> np.ndarray:
    """[world, n_waves] energies per rank and wave (for balance checks and gather layouts)."""
    out = np.zeros((world, len(n_E_per_wave)), dtype=np.int64)
    for r in range(world):
        for p, n in enumerate(n_E_per_wave):
            out[r, p] = energy_indices(int(n), p, r, world, block).size
    return out


def scatter_into(R_full: np.ndarray, idx: np.ndarray, R_part: np.ndarray) -> None:
    """Place a rank's [len(idx), C, C] slice into the wave's full [n_E, C, C] array (the optional
    gather a consumer of all R would do; not on the hot path)."""
    if R_part.shape[0] != idx.size:
        raise ValueError("slice and index lengths differ")
    R_full[idx] = R_part


def max_over_ranks(value: float, device="cpu") -> float:
    """MAX of a per-rank scalar (timings are reported as the slowest rank's).  A no-op without a
    process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
