"""Data-parallel schedules around the fused path: host plumbing only, no arithmetic.

Data (and context) parallelism replicates the weight, rank r holds a PARTIAL gradient G^(r), and an update that is
nonlinear in G -- AdamW's v is quadratic -- must wait for G = sum_r G^(r) (Prop. 2(ii)).  The paper's
answer is the bucket-transient schedule (304): weight-gradient tiles stream into a small ROTATING fp32
bucket, the bucket is all-reduced, the standalone update runs from the reduced bucket (a complete gradient for its
rows: Prop. 1 applies bucket-wise), and the bucket is recycled.  The transient is O(bucket), not O(parameters).
`BucketPlan` cuts a layer into row ranges that fit a bucket; `bucket_step_adamw` runs the schedule with the
all-reduce of bucket b in flight while bucket b + 1 is produced.

An update that is AFFINE in G needs no bucket (Prop. 2(iii); "reduce-into-state"):
`reduce_into_state` passes mu on exactly one rank and 0 on the others to B <- mu*B + dY^T X and all-reduces B in place.

The kernels are the library's (`forge_wgrad_store_g_grouped`, `forge_wgrad_accumulate_grouped`,
`forge_adamw_from_g`); the collective is torch.distributed's (NCCL over NVLink on GPUs).  The three steps are
injectable so that the schedule itself -- bucket cutting, slot rotation, ordering, the zero seed -- is covered by
world-size-2 gloo tests on CPU, where the tests supply the steps; the defaults call the CUDA binding and nothing else.
"""
from __future__ import annotations

from dataclasses import dataclass

ROW_ALIGN = 128           # bucket pieces start on a tile row block
DEFAULT_BUCKET_BYTES = 256 << 20


@dataclass(frozen=True)
class Piece:
    """Rows [r0, r1) of problem `p`; its fp32 gradient lives at [offset, offset + (r1 - r0) * in) of the bucket."""
    p: int
    r0: int
    r1: int
    offset: int
    cols: int

    @property
    def elems(self) -> int:
        return (self.r1 - self.r0) * self.cols


class BucketPlan:
    """Cuts problems [(out, in), ...] into buckets of at most `bucket_bytes` of fp32 gradient.

    A problem larger than a bucket is split into ROW_ALIGN-aligned row ranges (a row range of a layer is a problem of
    its own for the library: W / m / v row slices are contiguous, dY's column slice goes in through lddy); a bucket is
    never smaller than ROW_ALIGN rows of the widest problem.  `slots` buffers rotate ("recycled")."""

    def __init__(self, shapes, bucket_bytes: int = DEFAULT_BUCKET_BYTES, slots: int = 2):
        if slots < 1:
            raise ValueError("slots >= 1")
        shapes = [(int(o), int(i)) for o, i in shapes]
        cap = max(int(bucket_bytes) // 4, max(ROW_ALIGN * i for _, i in shapes))
        self.shapes, self.slots, self.capacity_elems = shapes, slots, cap
        self.buckets: list[list[Piece]] = []
        cur: list[Piece] = []
        used = 0
        for p, (out, cols) in enumerate(shapes):
            r = 0
            while r < out:
                room_rows = ((cap - used) // cols) // ROW_ALIGN * ROW_ALIGN
                if room_rows == 0:                      # bucket full: close it
                    self.buckets.append(cur)
                    cur, used = [], 0
                    continue
                r1 = min(out, r + room_rows)
                cur.append(Piece(p, r, r1, used, cols))
                used += (r1 - r) * cols
                r = r1
        if cur:
            self.buckets.append(cur)
        self.slot_elems = max(sum(pc.elems for pc in b) for b in self.buckets)

    @property
    def transient_bytes(self) -> int:
        """fp32 gradient memory the schedule holds: slots x the largest bucket, independent of the parameter count."""
        return self.slots * self.slot_elems * 4


def piece_problem(problem: dict, pc: Piece, G) -> dict:
    """The library problem for one piece: X whole, dY's column slice (a view), m = the piece's slice of the bucket."""
    return {"X": problem["X"], "dY": problem["dY"][:, pc.r0:pc.r1],
            "m": G[pc.offset:pc.offset + pc.elems].view(pc.r1 - pc.r0, pc.cols)}


def piece_state(problem: dict, pc: Piece) -> dict:
    """Row slices of W, m, v (and the int8 block scales) the update of one piece touches: views, updated in place."""
    return {k: problem[k][pc.r0:pc.r1] for k in ("W", "m", "v", "m_scale", "v_scale") if problem.get(k) is not None}


# ------------------------------------------------------------------------------------------------
# the three steps of the schedule; the defaults are the CUDA library and torch.distributed
# ------------------------------------------------------------------------------------------------
def _cuda_wgrad(piece_problems, first: bool):
    from . import binding as fb
    if first:
        fb.forge_wgrad_store_g_grouped(piece_problems)             # G = dY^T X
    else:
        fb.forge_wgrad_accumulate_grouped(piece_problems, 1.0, fb.FP32)   # later micro-batches: G <- 1*G + dY^T X


def _cuda_update(G2d, state: dict, step: int, hp: tuple):
    from . import binding as fb
    fb.forge_adamw_from_g(G2d, state["W"], state["m"], state["v"], step, *hp,
                          m_scale=state.get("m_scale"), v_scale=state.get("v_scale"))


def _cuda_accumulate(problems, mu: float, state_dtype):
    from . import binding as fb
    fb.forge_wgrad_accumulate_grouped(problems, mu, fb.FP32 if state_dtype is None else state_dtype)


def _all_reduce_async(t, group):
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return None
    return dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group, async_op=True)


def _micro_batches(problem: dict):
    X, dY = problem["X"], problem["dY"]
    if isinstance(X, (list, tuple)):
        if len(X) != len(dY) or not X:
            raise ValueError("X and dY must list the same micro-batches")
        return [dict(problem, X=x, dY=y) for x, y in zip(X, dY)]
    return [problem]


def bucket_step_adamw(problems, step: int, hp: tuple, plan: BucketPlan, pool, group=None, wgrad=None, update=None):
    """One data-parallel AdamW step of a layer by the bucket-transient schedule (304).

    problems: dicts with W, m, v (, m_scale, v_scale) and X, dY -- a tensor each, or a list of micro-batches, which are
    summed into the bucket before it is reduced (the exact-accumulation mode).  hp = (lr, beta1, beta2, eps, wd).
    pool: `plan.slots` fp32 buffers of >= plan.slot_elems elements on the problems' device.  The sum over ranks is
    what the update sees (no division: scale the loss).  On CUDA everything is enqueued on the current stream; the
    all-reduce of bucket b runs on the collective's own stream while bucket b + 1 is produced."""
    wgrad = _cuda_wgrad if wgrad is None else wgrad
    update = _cuda_update if update is None else update
    if len(pool) < plan.slots or any(g.numel() < plan.slot_elems for g in pool):
        raise ValueError("pool smaller than the plan")
    mbs = [_micro_batches(p) for p in problems]
    n_mb = len(mbs[0])
    if any(len(m) != n_mb for m in mbs):
        raise ValueError("every problem must carry the same number of micro-batches")
    pending = []                                           # (bucket, buffer, collective handle), oldest first

    def finish(entry):
        bucket, G, work = entry
        if work is not None:
            work.wait()                                    # on CUDA: the current stream waits, the host does not
        for pc in bucket:
            update(G[pc.offset:pc.offset + pc.elems].view(pc.r1 - pc.r0, pc.cols), piece_state(problems[pc.p], pc), step, hp)

    for b, bucket in enumerate(plan.buckets):
        if len(pending) == plan.slots:                     # the slot about to be overwritten must have been consumed
            finish(pending.pop(0))
        G = pool[b % plan.slots]
        for k in range(n_mb):
            wgrad([piece_problem(mbs[pc.p][k], pc, G) for pc in bucket], k == 0)
        used = sum(pc.elems for pc in bucket)
        pending.append((bucket, G, _all_reduce_async(G[:used], group)))
    while pending:
        finish(pending.pop(0))


def reduce_into_state(problems, mu: float, group=None, seed_rank: int = 0, state_dtype=None, accumulate=None):
    """B <- mu*B + sum_r dY_r^T X_r with no gradient and no bucket (Prop. 2(iii); 304): the rank
    `seed_rank` of the group passes mu, every other rank 0, and B (problem["m"]) is all-reduced in place.  B must be
    finite on every rank (0 * Inf is NaN); exact, not bit-exact: a reduction tree is not a sequential sum."""
    import torch.distributed as dist
    accumulate = _cuda_accumulate if accumulate is None else accumulate
    multi = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    rank = dist.get_rank(group) if multi else seed_rank
    accumulate(problems, float(mu) if rank == seed_rank else 0.0, state_dtype)
    works = [_all_reduce_async(p["m"], group) for p in problems]
    for w in works:
        if w is not None:
            w.wait()
