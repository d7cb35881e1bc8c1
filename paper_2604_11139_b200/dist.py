"""Band-sharded multi-GPU layer over libpwham -- one process per GPU, torch.distributed for the
plumbing (NCCL over NVLink / NVSwitch on a B200 node, gloo in the CPU tests).

The paper's two wave-function distributions (section 2.3 and Figure 1):
  * column-distributed: every process holds a contiguous range of BANDS with all plane waves -- what the Hamiltonian
    application, the Chebyshev filter and the density need; bands never interact there, so those steps
    run on the local block with no communication at all;
  * row-distributed: every process holds a contiguous range of PLANE WAVES with all bands, "as uniformly as possible" -- what the
    products A^H B of the Rayleigh-Ritz / orthogonalisation steps need: each process multiplies its row shard and the partial
    M x M matrices are summed (mpi-R; buffer 16 M^2 bytes, Table 2).
Switching between the two is one all-to-all-v (mpi-A; 16 N M / p bytes per process, Table 1).

A block is a (nband_local, npw) complex128 tensor in the column layout and a (nband, nrow_local) tensor in the row layout (rows of
the tensor are bands, as everywhere in this package).  Every arithmetic step is a libpwham kernel called through `binding`; this
module only moves data (pack, all-to-all, all-reduce) and keeps the ownership ranges.  `local_gram` / `local_rotate` can be
replaced by the caller (the CPU tests inject stand-ins, because libpwham has no CPU path).

Design note: on NVSwitch the all-to-all is bandwidth-symmetric, so the transposition is a single
`all_to_all_single` with uneven splits and the M x M reduction a single `all_reduce`; a Gram kernel that reads the peers' row
shards through NVLink peer mappings tile by tile (no staging copy) is the fused form of the same data flow and is not built
here -- it cannot be exercised on the one-GPU boxes this project is measured on.
"""
from __future__ import annotations

from typing import Callable, Optional, Tuple

import torch
import torch.distributed as dist


def split_range(n: int, p: int, r: int) -> Tuple[int, int]:
    """[lo, hi) of part r when n items are cut into p contiguous parts as uniformly as possible: the first n % p parts hold
    one item more."""
    q, rem = divmod(int(n), int(p))
    lo = r * q + min(r, rem)
    return lo, lo + q + (1 if r < rem else 0)


class BandSharded:
    """Ownership ranges and collectives of one k-point's wave functions, `nband` bands x `npw` plane waves, over a process group."""

    def __init__(self, nband: int, npw: int, group=None):
        self.group = group
        self.world = dist.get_world_size(group) if dist.is_initialized() else 1
        self.rank = dist.get_rank(group) if dist.is_initialized() else 0
        self.nband, self.npw = int(nband), int(npw)
        self.band_ranges = [split_range(nband, self.world, r) for r in range(self.world)]
        self.row_ranges = [split_range(npw, self.world, r) for r in range(self.world)]

    # ---- ownership ------------------------------------------------------------------------------------------------
    @property
    def bands(self) -> Tuple[int, int]:
        return self.band_ranges[self.rank]

    @property
    def rows(self) -> Tuple[int, int]:
        return self.row_ranges[self.rank]

    @property
    def nband_local(self) -> int:
        lo, hi = self.bands
        return hi - lo

    @property
    def nrow_local(self) -> int:
        lo, hi = self.rows
        return hi - lo

    def alltoall_bytes(self) -> int:
        """Bytes this process sends in one transposition (Table 1: 16 N M / p, minus the part it keeps)."""
        return 16 * self.nband_local * (self.npw - self.nrow_local)

    # ---- mpi-A: the two transpositions ----------------------------------------------------------------------------
    def to_rows(self, x_cols: torch.Tensor) -> torch.Tensor:
        """Column layout (nband_local, npw) -> row layout (nband, nrow_local)."""
        assert x_cols.shape == (self.nband_local, self.npw), (tuple(x_cols.shape), self.nband_local, self.npw)
        if self.world == 1:
            return x_cols.contiguous()
        # chunk r of the send buffer: my bands restricted to the rows of rank r, contiguous (nband_local x nrow_r)
        send = torch.cat([x_cols[:, lo:hi].reshape(-1) for lo, hi in self.row_ranges])
        in_splits = [self.nband_local * (hi - lo) for lo, hi in self.row_ranges]
        out_splits = [(hi - lo) * self.nrow_local for lo, hi in self.band_ranges]
        recv = torch.empty(self.nband * self.nrow_local, dtype=x_cols.dtype, device=x_cols.device)
        self._all_to_all(recv, send, out_splits, in_splits)
        # chunk s of the receive buffer is (nband_s x nrow_local): the chunks stacked in rank order ARE the row layout
        return recv.view(self.nband, self.nrow_local)

    def to_cols(self, x_rows: torch.Tensor) -> torch.Tensor:
        """Row layout (nband, nrow_local) -> column layout (nband_local, npw)."""
        assert x_rows.shape == (self.nband, self.nrow_local), (tuple(x_rows.shape), self.nband, self.nrow_local)
        if self.world == 1:
            return x_rows.contiguous()
        send = x_rows.contiguous().view(-1)             # bands of rank s are the contiguous chunk s
        in_splits = [(hi - lo) * self.nrow_local for lo, hi in self.band_ranges]
        out_splits = [self.nband_local * (hi - lo) for lo, hi in self.row_ranges]
        recv = torch.empty(self.nband_local * self.npw, dtype=x_rows.dtype, device=x_rows.device)
        self._all_to_all(recv, send, out_splits, in_splits)
        out = torch.empty((self.nband_local, self.npw), dtype=x_rows.dtype, device=x_rows.device)
        off = 0
        for lo, hi in self.row_ranges:                  # chunk r: my bands on the rows of rank r
            n = self.nband_local * (hi - lo)
            out[:, lo:hi] = recv[off:off + n].view(self.nband_local, hi - lo)
            off += n
        return out

    def _all_to_all(self, recv, send, out_splits, in_splits):
        # complex128 travels as pairs of float64 (NCCL has no complex type); splits are counted in complex elements
        r, s = torch.view_as_real(recv).view(-1), torch.view_as_real(send).view(-1)
        dist.all_to_all_single(r, s, [2 * v for v in out_splits], [2 * v for v in in_splits], group=self.group)

    # ---- mpi-R: products over row-distributed data ----------------------------------------------------------------
    def gram(self, x_cols: torch.Tensor, y_cols: torch.Tensor, local_gram: Optional[Callable] = None) -> torch.Tensor:
        """G = X^H Y (nband x nband, replicated on every rank) for column-distributed X, Y: two transpositions, the local
        product of the row shards (pwh_gram), one all-reduce of 16 M^2 bytes.  The partial product of a row shard is not
        Hermitian even when G is, so the general kernel is used."""
        return self.gram_rows(self.to_rows(x_cols), self.to_rows(y_cols), local_gram)

    def gram_rows(self, x_rows: torch.Tensor, y_rows: torch.Tensor, local_gram: Optional[Callable] = None) -> torch.Tensor:
        if local_gram is None:
            from . import binding
            local_gram = binding.gram
        if self.nrow_local > 0:
            g = local_gram(x_rows, y_rows).contiguous()
        else:
            g = torch.zeros((x_rows.shape[0], y_rows.shape[0]), dtype=x_rows.dtype, device=x_rows.device)
        if self.world > 1:
            dist.all_reduce(torch.view_as_real(g), op=dist.ReduceOp.SUM, group=self.group)
        return g

    def rotate(self, x_cols: torch.Tensor, q: torch.Tensor, local_rotate: Optional[Callable] = None) -> torch.Tensor:
        """Psi <- Psi Q for a replicated Q (nband x nband): the rotation mixes bands, so it runs on the row shards
        (pwh_rotate) between two transpositions (Algorithm 5 steps 4-5)."""
        if local_rotate is None:
            from . import binding
            local_rotate = binding.rotate
        rows = self.to_rows(x_cols)
        if self.nrow_local > 0:
            rows = local_rotate(rows, q)
        return self.to_cols(rows.contiguous())

    # ---- mpi-sR: small reductions ---------------------------------------------------------------------------------
    def minmax(self, local_min: float, local_max: float, device="cpu") -> Tuple[float, float]:
        """The 16-byte reduction of the Rayleigh-quotient bounds."""
        t = torch.tensor([-float(local_min), float(local_max)], dtype=torch.float64, device=device)
        if self.world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX, group=self.group)
        return -float(t[0]), float(t[1])

    def gather_band_values(self, local_vals: torch.Tensor) -> torch.Tensor:
        """Eigenvalues / residual norms of all bands from the per-rank pieces (16 M bytes)."""
        if self.world == 1:
            return local_vals.clone()
        out = torch.zeros(self.nband, dtype=local_vals.dtype, device=local_vals.device)
        lo, hi = self.bands
        out[lo:hi] = local_vals
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=self.group)
        return out

    # ---- steps that need no communication on the column layout ------------------------------------------------------
    def cheb_filter(self, ham, psi_cols: torch.Tensor, degree: int, a: float, b: float, a0: float) -> torch.Tensor:
        from . import binding
        return binding.cheb_filter(ham, psi_cols, degree, a, b, a0) if self.nband_local > 0 else psi_cols

    def apply_h(self, ham, psi_cols: torch.Tensor) -> torch.Tensor:
        from . import binding
        return binding.apply_h(ham, psi_cols) if self.nband_local > 0 else torch.empty_like(psi_cols)

    def density(self, ham, psi_cols: torch.Tensor, occ_all: torch.Tensor, rho: torch.Tensor, weight: float = 1.0,
                local_density: Optional[Callable] = None) -> torch.Tensor:
        """Adds this rank's bands to its PRIVATE partial density rho (pwh_density_accumulate on the local block; Algorithm 3
        steps 9-10).  After the last k-point `reduce_density` sums the partial arrays of all ranks."""
        if local_density is None:
            from . import binding
            local_density = binding.density_accumulate
        lo, hi = self.bands
        if hi > lo:
            local_density(ham, psi_cols, occ_all[lo:hi], rho, weight)
        return rho

    def reduce_density(self, rho: torch.Tensor) -> torch.Tensor:
        """One all-reduce of 8 F bytes: every rank ends with the density of all bands (and of all k-points accumulated so far)."""
        if self.world > 1:
            dist.all_reduce(rho, op=dist.ReduceOp.SUM, group=self.group)
        return rho
