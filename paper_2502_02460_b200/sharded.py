"""Steps 2, 3 and the back-transformation sharded over the GPUs of one NVSwitch domain
(the paper's multi-GPU direction, PAPER.md:118, PAPER.md:138;
DESIGN.md section 9).

One process per GPU.  Every rank holds H, S.  Step 1, two forms: chol="leading" -- every rank forms the part of
U it needs itself: the leading principal blocks of a Cholesky factor nest, chol(S[:k,:k]) = U[:k,:k], and a rank
that owns columns up to k needs no more than that block (gs_cholesky_leading; the same kernels give the same bits
on every rank; the last rank factors all of S) -- or chol="sharded" (push exchange with device-side ordering
only) -- gs_cholesky_sharded: the panels are dealt round-robin over the ranks, the owner's factored diagonal block
and every rank's pieces of the row panel are stored into all ranks, the trailing update of a panel's block columns
is its owner's.  After that the work is split by COLUMN RANGES, which need no exchange while they are formed:

    rank r owns the block columns J_r = [c_r, c_{r+1}) of U^-1, of G = T U^-1 and of H~
      1. V[:, J_r]  = (U^-1)[:, J_r]                (gs_invert_triangular_cols)
      2. G[:, J_r]  = T V[:, J_r]                   (gs_to_standard_g_cols)
      3. exchange: every rank gets every slab V[:, J_s], G[:, J_s]  -- the ONE exchange step
      4. H~[:, J_r] = V^H G[:, J_r] + G^H V[:, J_r], upper part      (gs_to_standard_cols)
    and, once the eigenvectors C~ of H~ are known (off the path), rank r forms the eigenvector
    columns K_r of C = V C~ (gs_backtransform_cols).

A column range of a column-major matrix is one contiguous slab.  Two forms of the exchange:
  exchange="push" (the GPU default): FUSED into the producing kernels.  The other ranks' buffers are mapped
      over NVLink/NVSwitch peer memory (CUDA IPC) and registered as push targets of the plan; the
      epilogues of the column-range kernels store every tile they produce into all of them (posted
      remote stores), so the slabs travel while the rest of the range is still being computed.  Steps 1-2
      and step 3 are then ordered either on the host (sync="host": stream synchronise + barrier) or ON THE
      DEVICE (sync="device"): every rank owns 2 x world 32-bit flags, mapped into its peers like the buffers;
      behind its producing kernels a rank writes the round's epoch into its "ready" slot of every peer
      (gs_exchange_signal) and its consuming launch waits until all ready slots of its own array carry the
      epoch (gs_exchange_wait) -- stream memory operations, no spinning kernel, no host round trip between
      producing and consuming; a second set of slots ("done") keeps a round's stores behind the previous
      round's reads.
  exchange="collective": an all-gather of unequal slabs after the kernels (one broadcast per owner;
      NCCL on the GPUs, gloo in the CPU test of this host logic) -- the baseline form.
With x = (c/N)^3, a range [c0, c1) costs kappa x1 (its leading Cholesky) + (x1 - x0) (steps 2-3: the cost
of column c grows like c^2 in all of them); the ranges are cut so that every rank carries the same sum
(column_ranges; kappa = time of step 1 / time of steps 2-3 on one GPU, 0.30 measured at N = 16384).

This module is host logic only: ranges, the order of the calls, the exchange.  All arithmetic runs
in libgs through the `plan` object (gs.Plan); there is no other implementation behind it.
"""
from __future__ import annotations

from dataclasses import dataclass

import torch
import torch.distributed as dist

from .workloads import colmajor_empty, colmajor_zeros


CHOL_WEIGHT = 0.30   # step 1 / (steps 2 + 3) on one GPU: 50.4 ms / 167.6 ms at N = 16384 (profiles/r01f_bench.json.txt)


def column_ranges(N: int, world: int, block: int, chol_weight: float = CHOL_WEIGHT) -> list[tuple[int, int]]:
    """[(c0, c1)] per rank: contiguous, covering [0, N), boundaries on multiples of `block` (the last
    ends at N).  With x = (c/N)^3 rank r carries chol_weight * x1 + (x1 - x0) (range_cost); equal sums
    give x1_r = (1 - rho^(r+1)) / (1 - rho^world), rho = 1 / (1 + chol_weight) (chol_weight = 0: the
    plain cube rule x1_r = (r+1)/world).  Ranks may get an empty range when there are fewer blocks
    than ranks."""
    if N <= 0 or world <= 0 or block <= 0 or chol_weight < 0:
        raise ValueError("N, world and block must be positive")
    nblk = (N + block - 1) // block
    rho = 1.0 / (1.0 + chol_weight)
    cuts = [0]
    for r in range(1, world):
        x = r / world if chol_weight == 0 else (1.0 - rho ** r) / (1.0 - rho ** world)
        b = round(nblk * x ** (1.0 / 3.0))
        cuts.append(min(max(b, cuts[-1]), nblk))
    cuts.append(nblk)
    return [(min(cuts[r] * block, N), min(cuts[r + 1] * block, N)) for r in range(world)]


def even_ranges(n: int, world: int, align: int = 1) -> list[tuple[int, int]]:
    """[(k0, k1)] per rank for work that costs the same per column (the back-transformation):
    equal shares, boundaries on multiples of `align`."""
    if n < 0 or world <= 0 or align <= 0:
        raise ValueError("bad arguments")
    units = (n + align - 1) // align
    cuts = [min(((units * r) // world) * align, n) for r in range(world)] + [n]
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def range_cost(c0: int, c1: int, N: int, chol_weight: float = CHOL_WEIGHT) -> float:
    """Relative cost of owning [c0, c1): its leading Cholesky plus its share of steps 2-3, in units of
    the one-GPU time of steps 2-3."""
    x0, x1 = (float(c0) / N) ** 3, (float(c1) / N) ** 3
    return (chol_weight * x1 if c1 > c0 else 0.0) + (x1 - x0)


def slab(X: torch.Tensor, c0: int, c1: int) -> torch.Tensor:
    """Columns [c0, c1) of a column-major matrix as a CONTIGUOUS (c1-c0) x rows tensor (a view)."""
    v = X.t()[c0:c1]
    if not v.is_contiguous():
        raise ValueError("expected a column-major matrix")
    return v


def exchange_slabs(mats, ranges, rank: int, world: int, group=None) -> None:
    """All-gather of unequal column slabs, in place: on return every rank holds columns J_s of every
    matrix in `mats` as formed by their owner s.  One broadcast per (owner, matrix)."""
    if world == 1:
        return
    for s, (c0, c1) in enumerate(ranges):
        if c1 <= c0:
            continue
        for X in mats:
            v = slab(X, c0, c1)
            if X.is_complex():
                v = torch.view_as_real(v)
            dist.broadcast(v, src=dist.get_global_rank(group, s) if group is not None else s, group=group)


@dataclass
class ShardedResult:
    U: torch.Tensor          # the leading cols[1] x cols[1] block holds U (all of U on the last rank); the rest is still S
    Uinv: torch.Tensor       # complete on every rank after the exchange
    G: torch.Tensor          # complete on every rank after the exchange
    Htilde: torch.Tensor     # upper triangle; only the columns of `cols` are valid before gather_htilde()
    cols: tuple[int, int]
    Uinv_work: torch.Tensor | None = None   # push mode: the rank's private work buffer of step 2
    C: torch.Tensor | None = None           # push mode: the registered N x nev back-transform result


class PeerMap:
    """Push mode: exchanges CUDA IPC handles of the ranks' buffers over the process group, maps the
    peers' allocations into this process and registers them as push targets of the plan."""

    def __init__(self, plan, rank: int, world: int, group=None):
        self.plan, self.rank, self.world, self.group = plan, rank, world, group
        self._bases = {}     # (owner rank, IPC handle) -> base pointer of the mapping (an allocation is mapped once)

    def map_all(self, local: torch.Tensor) -> list:
        """Device pointers, valid in this process, of the buffer every rank passes here (own rank: the local one)."""
        from . import gs
        mine = gs.ipc_export(local)
        infos = [None] * self.world
        dist.all_gather_object(infos, mine, group=self.group)
        ptrs = []
        for s, (handle, off) in enumerate(infos):
            if s == self.rank:
                ptrs.append(local.data_ptr())
                continue
            if (s, handle) not in self._bases:
                self._bases[(s, handle)] = gs.ipc_open(handle, 0)
            ptrs.append(self._bases[(s, handle)] + off)
        return ptrs

    def register(self, kind: int, local: torch.Tensor, include_self: bool) -> None:
        ptrs = self.map_all(local)
        if not include_self:
            ptrs = [p for s, p in enumerate(ptrs) if s != self.rank]
        self.plan.set_push_targets(kind, ptrs)

    def close(self) -> None:
        from . import gs
        for kind in range(4):
            self.plan.set_push_targets(kind, [])
        for base in self._bases.values():
            gs.ipc_close(base, 0)
        self._bases = {}


class ShardedReduction:
    """Host driver of the sharded path for one rank.  `plan` is a gs.Plan (or, in the CPU test of this
    host logic, an object with the same column-range methods -- exchange="collective" only)."""

    def __init__(self, plan, rank: int = 0, world: int = 1, group=None, exchange: str = "collective", sync: str = "host",
                 chol: str = "leading"):
        if exchange not in ("collective", "push"):
            raise ValueError("exchange must be 'collective' or 'push'")
        if sync not in ("host", "device"):
            raise ValueError("sync must be 'host' or 'device'")
        if chol not in ("leading", "sharded"):
            raise ValueError("chol must be 'leading' (every rank factors the leading block it needs) or 'sharded' "
                             "(gs_cholesky_sharded: panels dealt round-robin over the ranks)")
        if chol == "sharded" and world > 1 and not (exchange == "push" and sync == "device"):
            raise ValueError("chol='sharded' stores into the peers' buffers and orders itself by device-side flags: "
                             "it needs exchange='push' and sync='device'")
        if chol == "sharded" and world > 8:
            raise ValueError("chol='sharded': at most 8 ranks (one NVSwitch domain)")
        self.plan = plan
        self.rank, self.world, self.group = int(rank), int(world), group
        self.push = exchange == "push" and self.world > 1
        self.device_sync = self.push and sync == "device"
        self.chol_sharded = chol == "sharded" and self.world > 1
        self.chol_epoch = 0
        self.U_ptrs = self.ws_ptrs = self.chol_flags = self.chol_flag_ptrs = None
        self.epoch = 0
        self.flags = None            # int32[2 * world]: ready slots, then done slots (device sync)
        self.flag_ptrs = None        # this rank's view of every rank's flag array
        self.N, self.nev = plan.N, plan.nev
        # (chol='sharded': step 1 costs every rank the same, whatever its columns -- the plain cube rule balances steps 2-3)
        self.ranges = column_ranges(self.N, self.world, plan.block, 0.0 if chol == "sharded" and self.world > 1 else CHOL_WEIGHT)
        self.eig_ranges = even_ranges(self.nev, self.world, 2)
        self.peers = None

    def _barrier(self) -> None:
        if self.world > 1:
            dist.barrier(group=self.group)

    def _check_all(self, device, stream=None) -> None:
        """Synchronises this rank's stream and agrees on the numerical status over ALL ranks: a rank
        whose leading block is fine must not run on into an exchange that a failing rank never joins.
        Raises GsError(status, first bad pivot) on every rank alike: GS_ERR_NOT_POSDEF (a pivot of S that
        is not positive) or GS_ERR_SINGULAR (a zero on the diagonal of U in the column-range inversion)."""
        info = int(self.plan.last_info(stream=stream, raise_on_failure=False))
        # last_info reports |index|; the status says which failure it was (gs.h: gs_last_info)
        status = self.plan.last_status if hasattr(self.plan, "last_status") else (2 if info else 0)
        # one MIN reduction orders by pivot index first, then by status: key = 8 * index + status
        key = (8 * abs(info) + int(status)) if info else (1 << 62)
        if self.world > 1:
            on_cpu = dist.get_backend(self.group) == "gloo"
            t = torch.tensor([key], dtype=torch.int64, device="cpu" if on_cpu else device)
            dist.all_reduce(t, op=dist.ReduceOp.MIN, group=self.group)
            key = int(t.item())
        if key != (1 << 62):
            from .gs import GsError
            bad, status = key >> 3, key & 7
            what = "a zero on the diagonal of U" if status == 3 else "S is not positive definite"
            raise GsError(status or 2, bad, f"sharded reduction: {what} (first bad pivot over all ranks)")

    def alloc(self, like: torch.Tensor) -> ShardedResult:
        """The N x N result buffers of reduce() (so a loop of reductions allocates once).  Push mode:
        collective over the ranks -- also maps the peers' buffers and registers the push targets."""
        N = self.N
        U, Uinv, G = (colmajor_empty(N, N, dtype=like.dtype, device=like.device) for _ in range(3))
        Ht = colmajor_zeros(N, N, dtype=like.dtype, device=like.device)
        res = ShardedResult(U, Uinv, G, Ht, self.ranges[self.rank])
        if self.push:
            from . import gs
            if self.peers is not None:
                # a second alloc() would leak the first one's IPC mappings (and re-open handles the caching
                # allocator may hand out again): push mode works on ONE persistent result
                raise RuntimeError("push mode: alloc() was already called; pass out=<that result> to reduce(), "
                                   "or close() first")
            res.Uinv.zero_()               # exchange buffer: nothing is ever pushed below the diagonal
            res.Uinv_work = colmajor_empty(N, N, dtype=like.dtype, device=like.device)
            res.C = colmajor_empty(N, max(self.nev, 1), dtype=like.dtype, device=like.device)[:, :self.nev]
            torch.cuda.synchronize(like.device)
            self.peers = PeerMap(self.plan, self.rank, self.world, self.group)
            self.peers.register(gs.GS_PUSH_UINV, res.Uinv, include_self=True)
            self.peers.register(gs.GS_PUSH_G, res.G, include_self=False)
            self.peers.register(gs.GS_PUSH_HTILDE, res.Htilde, include_self=False)
            if self.nev > 0:
                self.peers.register(gs.GS_PUSH_C, res.C, include_self=False)
            if self.device_sync:
                self.flags = torch.zeros(2 * self.world, dtype=torch.int32, device=like.device)
                torch.cuda.synchronize(like.device)
                self.flag_ptrs = self.peers.map_all(self.flags)
                self.epoch = 0
            if self.chol_sharded:
                # step 1 over the ranks: the peers' U buffers and plan workspaces (the inverted diagonal blocks travel
                # through them) and a flag array of its own
                self.U_ptrs = self.peers.map_all(res.U)
                self.ws_ptrs = self.peers.map_all(self.plan.workspace)
                self.chol_flags = torch.zeros(self.world, dtype=torch.int32, device=like.device)
                torch.cuda.synchronize(like.device)
                self.chol_flag_ptrs = self.peers.map_all(self.chol_flags)
                self.chol_epoch = 0
            self._barrier()
        return res

    def close(self) -> None:
        """Push mode: collective; unmaps the peers' buffers (call before the buffers are freed)."""
        if self.peers is not None:
            torch.cuda.synchronize()
            self._barrier()
            self.peers.close()
            self.peers = None
            self._barrier()

    def reduce(self, H: torch.Tensor, S: torch.Tensor, stream=None, out: ShardedResult | None = None) -> ShardedResult:
        """Steps 1-3.  H, S: column-major N x N on this rank's device, identical on all ranks; S is not
        modified.  Returns this rank's columns of the upper triangle of H~ (and U, U^-1, G in full;
        push mode: H~ in full too, once every rank has returned and a barrier has passed)."""
        plan = self.plan
        res = self.alloc(H) if out is None else out
        if stream is not None and stream != torch.cuda.current_stream(H.device):
            # the torch-side operations below (the copy of S, NCCL broadcasts, all-reduces) run on torch's
            # CURRENT stream: make `stream` current so that they are ordered with the libgs kernels
            with torch.cuda.stream(stream):
                return self.reduce(H, S, stream=stream, out=res)
        c0, c1 = res.cols
        U, Uinv, G, Ht = res.U, res.Uinv, res.G, res.Htilde
        if self.device_sync:
            return self._reduce_device_sync(H, S, res, stream)
        if self.push:
            self._barrier()                # the peers have finished reading what the last round pushed
        work = res.Uinv_work if self.push else Uinv
        if c1 > c0:                        # (a rank without columns -- more ranks than blocks -- only takes part in the exchange)
            U.copy_(S)
            plan.cholesky_leading(U, c1, stream=stream)                       # the leading block this rank needs
            plan.invert_triangular_cols(U, work, c0, c1 - c0, stream=stream)  # push: slab -> every rank's Uinv
            plan.to_standard_g_cols(H, work, G, c0, c1 - c0, stream=stream)   # push: slab -> every other rank's G
        self._check_all(H.device, stream)                                 # synchronises: the slabs are final; all ranks agree
        if self.push:
            self._barrier()                # ... and have landed everywhere
        else:
            exchange_slabs((Uinv, G), self.ranges, self.rank, self.world, self.group)
        if c1 > c0:
            plan.to_standard_cols(Uinv, G, Ht, c0, c1 - c0, stream=stream)
        plan.last_info(stream=stream)
        return res

    def _slots(self, which: int):
        """(addresses of MY slot `which` (0 ready, 1 done) in every rank's flag array, addresses of all ranks' slots in mine)"""
        w, r = self.world, self.rank
        mine_everywhere = [p + 4 * (which * w + r) for p in self.flag_ptrs]
        all_in_mine = [self.flag_ptrs[r] + 4 * (which * w + s) for s in range(w)]
        return mine_everywhere, all_in_mine

    def _reduce_device_sync(self, H, S, res, stream):
        """reduce() with the producing and the consuming launches ordered by device-side flags: nothing between
        step 2 and step 3 waits for the host.  Every rank signals, whatever its own numerical status (a failed rank's
        compute calls are no-ops; its signals are not), so no stream waits for ever; the status is agreed at the end."""
        plan = self.plan
        c0, c1 = res.cols
        self.epoch += 1
        e = self.epoch
        ready_out, ready_in = self._slots(0)
        done_out, done_in = self._slots(1)
        if e > 1:
            plan.exchange_wait(done_in, e - 1, stream=stream)     # the peers have read what the last round pushed
        if self.chol_sharded:
            # every rank takes part (it owns panels whatever its column range) and ends up with ALL of U
            res.U.copy_(S)
            plan.cholesky_sharded(res.U, self.rank, self.world, self.U_ptrs, self.ws_ptrs, self.chol_flag_ptrs,
                                  epoch0=self.chol_epoch, stream=stream)
            self.chol_epoch += plan.cholesky_sharded_epochs()
        elif c1 > c0:
            res.U.copy_(S)
            plan.cholesky_leading(res.U, c1, stream=stream)
        if c1 > c0:
            plan.invert_triangular_cols(res.U, res.Uinv_work, c0, c1 - c0, stream=stream)
            plan.to_standard_g_cols(H, res.Uinv_work, res.G, c0, c1 - c0, stream=stream)
        plan.exchange_signal(ready_out, e, stream=stream)          # behind the kernels whose epilogues pushed the slabs
        plan.exchange_wait(ready_in, e, stream=stream)             # every rank's slabs have landed here
        if c1 > c0:
            plan.to_standard_cols(res.Uinv, res.G, res.Htilde, c0, c1 - c0, stream=stream)
        plan.exchange_signal(done_out, e, stream=stream)           # ... and my columns of H~ are out as well
        self._check_all(H.device, stream)
        return res

    def gather_htilde(self, res: ShardedResult) -> torch.Tensor:
        """Every rank gets all columns of the upper triangle of H~ (for an off-path eigensolver)."""
        if self.device_sync:
            _, done_in = self._slots(1)
            self.plan.exchange_wait(done_in, self.epoch)           # step 3 of every rank has pushed its columns
        elif self.push:
            self._barrier()                # step 3 already pushed them
        else:
            exchange_slabs((res.Htilde,), self.ranges, self.rank, self.world, self.group)
        return res.Htilde

    def backtransform(self, Uinv: torch.Tensor, Ctilde: torch.Tensor, stream=None, out: torch.Tensor | None = None) -> torch.Tensor:
        """C = U^-1 C~, eigenvector columns split evenly over the ranks, then gathered.  Push mode:
        `out` must be the registered buffer (ShardedResult.C of alloc())."""
        if stream is not None and stream != torch.cuda.current_stream(Ctilde.device):
            with torch.cuda.stream(stream):   # see reduce(): the exchange runs on torch's current stream
                return self.backtransform(Uinv, Ctilde, stream=stream, out=out)
        C = colmajor_empty(self.N, self.nev, dtype=Ctilde.dtype, device=Ctilde.device) if out is None else out
        k0, k1 = self.eig_ranges[self.rank]
        if self.push and out is None:
            raise ValueError("push mode: pass out=res.C (the buffer whose peers are registered)")
        self.plan.backtransform_cols(Uinv, Ctilde, C, k0, k1 - k0, stream=stream)
        self.plan.last_info(stream=stream)
        if self.push:
            self._barrier()
        else:
            exchange_slabs((C,), self.eig_ranges, self.rank, self.world, self.group)
        return C
