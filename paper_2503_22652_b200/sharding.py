"""Host-side multi-GPU plumbing (one process per GPU, torch.distributed).  No method arithmetic here: the partition
is index bookkeeping, the exchange moves buffers, every number is produced by the library's kernels.

Two ways the filter shards:

* COLUMNS.  Algorithm 3 touches column j only through eps_j and Lambda_k[j], so ranks may own
  disjoint column shards of the block against a replica of the operator: no data-path collective (`column_shard`,
  `reduce_job`; bench.py --gpus N).

* ROWS (the paper's scheme: domain decomposition with nearest-neighbour exchange inside the matvec, optionally with
  BF16 on the wire, "TF32B").  `slab_partition_fe` cuts an FE mesh into slabs of cells along the
  slowest mesh direction; a rank owns its cells and every row they touch, so the node plane between two slabs is
  replicated on both ranks.  `RowShardedFilter` runs rchfsi_filter step by step and, after each step, exchanges one
  buffer per neighbour with the interface rows' share of the product (rchfsi_interface_save / _pack / _apply).
"""


def column_shard(n_cols, rank, world):
    """[lo, hi) of the global columns owned by `rank`: contiguous, disjoint, covering, sizes differ by <= 1."""
    if world < 1 or not 0 <= rank < world or n_cols < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_cols, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def reduce_job(ms_local, units_local, group=None):
    """(max over ranks of the local time, sum over ranks of the local unit count) via torch.distributed.
    Works on any backend (NCCL on GPUs, gloo in the CPU tests); world size 1 needs no process group."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(ms_local), float(units_local)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=dev)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    dist.all_reduce(u, op=dist.ReduceOp.SUM, group=group)
    return float(t.item()), float(u.item())


# ------------------------------------------------------------------------------------------------ row slabs
def slab_partition_fe(prob, rank, world):
    """Slab `rank` of `world` of an FE workload dict (workloads.fe_problem numbering: cell c = (cx*nc + cy)*nc + cz,
    node g = ((gx*ng + gy)*ng + gz), ng = q*nc + 1).  Cells are cut along cx, so the rows of a slab are ONE contiguous
    range of global rows and the interface between slabs r and r+1 is the node plane gx = q * x1 (ng^2 rows).

    Returns a dict: the local problem (same keys as the workload: m, n_cells, n_loc, conn [local rows], A_cells, B_cell,
    dinv), plus row0 / row1 (global row range, both interface planes included), cells (global cell ids),
    if_lower / if_upper (LOCAL row ids of the interface planes, empty at the domain boundary)."""
    import numpy as np
    nc, q = int(prob["nc"]), int(prob["q"])
    if not 1 <= world <= nc or not 0 <= rank < world:
        raise ValueError("need 1 <= world <= cells per direction and 0 <= rank < world")
    ng = q * nc + 1
    x0, x1 = column_shard(nc, rank, world)            # cell layers [x0, x1) along x
    plane = ng * ng
    row0, row1 = q * x0 * plane, (q * x1 + 1) * plane
    cells = np.arange(x0 * nc * nc, x1 * nc * nc, dtype=np.int64)
    conn = (prob["conn"][cells].astype(np.int64) - row0).astype(np.int32)
    assert conn.min() == 0 and conn.max() == row1 - row0 - 1
    local = dict(kind="fe", m=row1 - row0, n_cells=len(cells), n_loc=prob["n_loc"], nc=nc, q=q, conn=conn,
                 A_cells=prob["A_cells"][cells], B_cell=prob["B_cell"], dinv=prob["dinv"][row0:row1],
                 row0=row0, row1=row1, cells=cells,
                 if_lower=np.arange(0, plane, dtype=np.int32) if rank > 0 else np.zeros(0, np.int32),
                 if_upper=np.arange(row1 - row0 - plane, row1 - row0, dtype=np.int32) if rank < world - 1
                 else np.zeros(0, np.int32))
    return local


def neighbor_exchange(send, recv, n_lo, n_hi, rank, group=None):
    """send[:n_lo] <-> rank-1 and send[n_lo:n_lo+n_hi] <-> rank+1 into the same slices of recv: one message per
    neighbour and direction (torch.distributed P2P; NCCL over NVLink for CUDA buffers, gloo for CPU buffers)."""
    import torch.distributed as dist
    ops = []
    lo, hi = n_lo, n_lo + n_hi
    if n_lo:
        ops += [dist.P2POp(dist.isend, send[:lo], rank - 1, group), dist.P2POp(dist.irecv, recv[:lo], rank - 1, group)]
    if n_hi:
        ops += [dist.P2POp(dist.isend, send[lo:hi], rank + 1, group), dist.P2POp(dist.irecv, recv[lo:hi], rank + 1, group)]
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()


WIRE_DTYPE = {"fp64": "float64", "fp32": "float32", "bf16": "bfloat16"}


class RowShardedFilter:
    """One rank's part of a row-sharded R-ChFSI filter (Algorithm 3, with the paper's nearest-neighbour
    exchange).  `solver` is an Rchfsi handle on this rank's slab (slab_partition_fe); `if_lower` /
    `if_upper` are the local rows shared with rank-1 / rank+1.  Per recurrence step ONE buffer of
    len(interface) x N wire-precision numbers goes to each neighbour and one comes back.

    `exchange(send_lower, send_upper, recv_lower, recv_upper)` moves the buffers; the default uses torch.distributed
    point-to-point calls between neighbouring ranks of `group` (NCCL over NVLink on GPUs).  Tests drive several shards
    in one process with `filter_in_process`."""

    def __init__(self, solver, if_lower, if_upper, wire="bf16", group=None, rank=None, world=None):
        import torch
        self.s = solver
        dev = torch.device("cuda", torch.cuda.current_device())
        self.n_lo, self.n_hi = int(len(if_lower)), int(len(if_upper))
        rows = torch.cat([torch.as_tensor(if_lower, dtype=torch.int32), torch.as_tensor(if_upper, dtype=torch.int32)])
        self.rows = rows.to(dev)
        self.wire = wire
        dt = getattr(torch, WIRE_DTYPE[wire])
        n = self.n_lo + self.n_hi
        self.send = torch.zeros((max(n, 1), solver.N), dtype=dt, device=dev)
        self.recv = torch.zeros((max(n, 1), solver.N), dtype=dt, device=dev)
        self.group, self.rank, self.world = group, rank, world
        self.bytes_per_step = n * solver.N * self.send.element_size()

    # ---- the three phases of one step (split so that an in-process driver can interleave several shards)
    def begin(self, X, ritz, G, degree, lam_min, lam_T, lam_max):
        from .binding import METHOD_RCHFSI
        self.s.filter_begin(METHOD_RCHFSI, X, ritz, G, degree, lam_min, lam_T, lam_max)

    def step_and_pack(self):
        if self.rows.numel():
            self.s.interface_save(self.rows)
        self.s.filter_step()
        if self.rows.numel():
            self.s.interface_pack(self.rows, self.wire, self.send)

    def apply(self):
        if self.rows.numel():
            self.s.interface_apply(self.rows, self.wire, self.send, self.recv)

    def exchange_distributed(self):
        neighbor_exchange(self.send, self.recv, self.n_lo, self.n_hi, self.rank, self.group)

    def filter(self, X, ritz, G, degree, lam_min, lam_T, lam_max):
        """This rank's rows of Y_p (X overwritten); every rank of the group must call it."""
        self.begin(X, ritz, G, degree, lam_min, lam_T, lam_max)
        while self.s.filter_steps_left() > 0:
            self.step_and_pack()
            self.exchange_distributed()
            self.apply()
        self.s.filter_end()
        return X


def exchange_in_process(shards):
    """The neighbour exchange for shards that live in ONE process (tests, single-GPU emulation): shard r's upper send
    buffer is shard r+1's lower receive buffer and vice versa."""
    for r in range(len(shards) - 1):
        a, b = shards[r], shards[r + 1]
        assert a.n_hi == b.n_lo
        a.recv[a.n_lo:a.n_lo + a.n_hi].copy_(b.send[:b.n_lo])
        b.recv[:b.n_lo].copy_(a.send[a.n_lo:a.n_lo + a.n_hi])


def filter_in_process(shards, blocks, degree, lam_min, lam_T, lam_max):
    """Run the row-sharded filter with all shards in this process, in lockstep.  blocks[r] = (X_r, ritz, G_r)."""
    for sh, (X, ritz, G) in zip(shards, blocks):
        sh.begin(X, ritz, G, degree, lam_min, lam_T, lam_max)
    while shards[0].s.filter_steps_left() > 0:
        for sh in shards:
            sh.step_and_pack()
        exchange_in_process(shards)
        for sh in shards:
            sh.apply()
    for sh in shards:
        sh.s.filter_end()
    return [b[0] for b in blocks]
