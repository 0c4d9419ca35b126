"""(k-point, band) sharding of the hot path across ranks -- SURVEY.md section 8(e) / 8(f) rank 4.

The paper distributes k-points over MPI processes ("MPI parallelisation over k-points"); inside a
k-point every band column of `HC` is independent, so `apply_H` shards over (k, band range) with NO collective.
Two operations do exchange data:

* the overlap / subspace matrix `M = C1^dagger O C2` with the bands of both operands sharded: every rank needs all
  rows of `C1` against its own columns `C2`.  `sharded_overlap` offers the two usual schedules --
  "allgather": ONE all-gather of `C1` over the band group, then one local GEMM (`jdft_overlap`);
  "ring": world-1 neighbour exchanges of one shard each, the GEMM on the shard that has arrived running while the
  next shard is in flight (the transfer hides behind DMMA time; peak extra memory is two shards, not nb rows).
  Either way rank r ends with the column block `M[:, lo_r:hi_r]`; `gather_columns` assembles the small
  nb x nb matrix on every rank when the caller wants it replicated.
* the density `n = sum_k w_k sum_b f_b |I C_b|^2`: a local `jdft_density` over the rank's bands, then ONE all-reduce
  (sum) of the N-point real field.

This module is process-group glue only (`torch.distributed`; NCCL on GPUs, gloo in the CPU tests): the arithmetic is
the library's (`binding.jdft_*`), passed in as `ops` so the host logic can be exercised on CPU ranks by the tests with
a stand-in.  The default `ops` is the CUDA binding and raises when libjdft_b200.so is missing -- no CPU fallback.
"""
import torch
import torch.distributed as dist


def shard_range(n, parts, index):
    """Contiguous balanced split of range(n) into `parts` pieces; the first n % parts pieces get one more."""
    if parts <= 0 or not 0 <= index < parts:
        raise ValueError("need 0 <= index < parts")
    q, r = divmod(n, parts)
    lo = index * q + min(index, r)
    return lo, lo + q + (1 if index < r else 0)


class KBLayout:
    """Which (k-point, band range) units rank `rank` of `world` owns.

    world <= nk: k-points are dealt out in contiguous balanced runs, each rank holds ALL bands of its k-points
    (the paper's layout, no band group, no collective in the overlap).
    world > nk: the ranks are split into nk contiguous groups (balanced); group g works on k-point g and shards the
    nb bands over its members.  `group_ranks` lists the ranks that share this rank's k-point(s)."""

    def __init__(self, nk, nb, world, rank):
        if nk < 1 or nb < 1 or world < 1 or not 0 <= rank < world:
            raise ValueError("bad layout arguments")
        self.nk, self.nb, self.world, self.rank = nk, nb, world, rank
        if world <= nk:
            klo, khi = shard_range(nk, world, rank)
            self.group_index = rank
            self.group_ranks = [rank]
            self.units = [(k, 0, nb) for k in range(klo, khi)]
        else:
            for g in range(nk):
                rlo, rhi = shard_range(world, nk, g)
                if rlo <= rank < rhi:
                    break
            self.group_index = g
            self.group_ranks = list(range(rlo, rhi))
            blo, bhi = shard_range(nb, rhi - rlo, rank - rlo)
            self.units = [(g, blo, bhi)] if bhi > blo else []
        self.group_size = len(self.group_ranks)
        self.group_rank = self.group_ranks.index(rank)

    def group_units(self):
        """Like `units`, but a member of a band group whose band range is empty still gets its (k, lo, lo) entry: it
        has to take part in the group's collectives."""
        if self.units or self.world <= self.nk:
            return list(self.units)
        blo, bhi = shard_range(self.nb, self.group_size, self.group_rank)
        return [(self.group_index, blo, bhi)]

    def band_ranges(self):
        """Band range of every member of this rank's group, in group order."""
        return [shard_range(self.nb, self.group_size, i) for i in range(self.group_size)]

    def new_band_group(self):
        """Creates the process groups of ALL k groups (a collective over the world, as `dist.new_group` requires)
        and returns this rank's; None when the group is this rank alone."""
        if self.world <= self.nk:
            return None
        mine = None
        for g in range(self.nk):
            rlo, rhi = shard_range(self.world, self.nk, g)
            grp = dist.new_group(list(range(rlo, rhi)))
            if g == self.group_index:
                mine = grp
        return mine


def _default_ops():
    from . import binding  # raises if the CUDA library is missing: there is no CPU path
    return binding


def sharded_apply_H(basis, Vloc, P, D, C_local, HC_local=None, ops=None):
    """`HC` for this rank's band columns: a local call, no collective (every column is independent)."""
    ops = ops or _default_ops()
    return ops.jdft_apply_H(basis, Vloc, P, D, C_local, HC_local)


def _group_info(group):
    if group is None and not dist.is_initialized():
        return 1, 0
    return dist.get_world_size(group), dist.get_rank(group)


def _global_rank(group, group_rank):
    return group_rank if group is None else dist.get_global_rank(group, group_rank)


def sharded_overlap(basis, C1_local, C2_local, nb, group=None, mode="allgather", subspace=False, ops=None):
    """Column block `M[:, lo:hi]` (all nb rows, this rank's columns) of `M[a, b] = Omega sum_n conj(C1[a, n]) C2[b, n]`
    (`subspace=True`: no Omega, `C2` is e.g. `HC`), with the nb rows of `C1` band-sharded over `group` by
    `shard_range(nb, size, rank)` and `C2_local` any band block of this rank.  mode: "allgather" | "ring"."""
    ops = ops or _default_ops()
    gemm = ops.jdft_subspace if subspace else ops.jdft_overlap
    size, me = _group_info(group)
    ranges = [shard_range(nb, size, i) for i in range(size)]
    lo, hi = ranges[me]
    if C1_local.shape[0] != hi - lo:
        raise ValueError("C1_local must hold rows %d:%d of C1 on group rank %d" % (lo, hi, me))
    nG = C1_local.shape[1]
    if size == 1:
        return gemm(basis, C1_local, C2_local)
    rows_max = ranges[0][1] - ranges[0][0]
    if mode == "allgather":
        # one collective: shards padded to the largest (they differ by at most one row), compacted only if ragged
        send = C1_local
        if send.shape[0] != rows_max:
            send = torch.zeros((rows_max, nG), dtype=C1_local.dtype, device=C1_local.device)
            send[: hi - lo] = C1_local
        full = torch.empty((size * rows_max, nG), dtype=C1_local.dtype, device=C1_local.device)
        dist.all_gather_into_tensor(torch.view_as_real(full), torch.view_as_real(send.contiguous()), group=group)
        if size * rows_max != nb:
            full = torch.cat([full[i * rows_max: i * rows_max + (r1 - r0)] for i, (r0, r1) in enumerate(ranges)])
        return gemm(basis, full, C2_local)
    if mode != "ring":
        raise ValueError("mode must be 'allgather' or 'ring'")
    # ring: at step s this rank holds the shard of group rank (me - s) % size; it forwards that shard to its right
    # neighbour and multiplies it while the transfer is in flight.
    right, left = _global_rank(group, (me + 1) % size), _global_rank(group, (me - 1) % size)
    cur = torch.zeros((rows_max, nG), dtype=C1_local.dtype, device=C1_local.device)
    cur[: hi - lo] = C1_local
    blocks = [None] * size
    for s in range(size):
        src = (me - s) % size
        reqs, nxt = [], None
        if s + 1 < size:
            nxt = torch.empty_like(cur)
            reqs = dist.batch_isend_irecv([dist.P2POp(dist.isend, torch.view_as_real(cur), right, group),
                                           dist.P2POp(dist.irecv, torch.view_as_real(nxt), left, group)])
        r0, r1 = ranges[src]
        if r1 > r0:
            blocks[src] = gemm(basis, cur[: r1 - r0], C2_local).clone()
        for q in reqs:
            q.wait()
        cur = nxt
    return torch.cat([b for b in blocks if b is not None], dim=0)


def gather_columns(M_cols, nb, group=None):
    """Assembles the replicated nb x nb matrix from the column blocks `sharded_overlap` leaves on each rank
    (one small all-gather; blocks padded to the widest)."""
    size, me = _group_info(group)
    if size == 1:
        return M_cols
    ranges = [shard_range(nb, size, i) for i in range(size)]
    wmax = ranges[0][1] - ranges[0][0]
    nrow = M_cols.shape[0]
    send = torch.zeros((wmax, nrow), dtype=M_cols.dtype, device=M_cols.device)
    send[: M_cols.shape[1]] = M_cols.t()
    full = torch.empty((size * wmax, nrow), dtype=M_cols.dtype, device=M_cols.device)
    dist.all_gather_into_tensor(torch.view_as_real(full), torch.view_as_real(send), group=group)
    return torch.cat([full[i * wmax: i * wmax + (r1 - r0)] for i, (r0, r1) in enumerate(ranges)]).t()


def sharded_density(basis, C_local, f_local, group=None, weight=1.0, n=None, ops=None):
    """`n(r) (+)= weight * sum_{b in this rank} f_b |I C_b|^2`, then ONE all-reduce (sum) over `group` (pass the world
    group to sum over k-points and bands at once; `weight` is the k-point weight).  Every rank returns the total."""
    ops = ops or _default_ops()
    size, _ = _group_info(group)
    if C_local.shape[0] > 0:
        part = ops.jdft_density(basis, C_local, f_local * weight)
    else:
        part = torch.zeros(tuple(basis.S), dtype=torch.float64, device=C_local.device)
    if size > 1:
        dist.all_reduce(part, op=dist.ReduceOp.SUM, group=group)
    if n is None:
        return part
    n += part.view_as(n)
    return n


def sharded_step(layout, kdata, Vloc, D, group=None, mode="allgather", overlap=True, ops=None):
    """One pass of the hot path over this rank's (k-point, band range) units -- what `bench.py --shard kb` times.
    `kdata[k] = dict(basis=..., P=..., C=<this rank's band rows of k-point k>, HC=<optional output>)`.
    Per unit: `HC` for the local band columns (no collective) and, with `overlap`, this rank's column block
    `M[:, lo:hi]` of `C^dagger O C` of that k-point (one all-gather or a ring over the band group).
    Returns `{k: (HC_local, M_cols or None)}`."""
    out = {}
    for k, blo, bhi in layout.group_units():
        d = kdata[k]
        HC = d["C"].new_zeros(d["C"].shape) if bhi == blo else sharded_apply_H(d["basis"], Vloc, d["P"], D, d["C"], d.get("HC"), ops=ops)
        M = None
        if overlap and layout.group_size == 1:      # this rank holds all bands of the k-point: a local GEMM, no collective
            M = (ops or _default_ops()).jdft_overlap(d["basis"], d["C"], d["C"])
        elif overlap:
            M = sharded_overlap(d["basis"], d["C"], d["C"], layout.nb, group=group, mode=mode, ops=ops)
        out[k] = (HC, M)
    return out
