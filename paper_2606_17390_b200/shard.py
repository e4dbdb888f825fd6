"""Row-ownership sharding of fem_assemble over several GPUs: one process per GPU, ONE collective.

Element evaluations are independent (the paper vmaps over them); the only coupling is the sum into shared
rows (Eq.(34)/(38) :253, :274).  Rank g owns a contiguous slab of nodes and therefore whole CSR rows; it evaluates every
element that touches one of its nodes (owned elements plus a one-element-thick ghost layer, recomputed on both sides), so
its rows are complete and no output is shared or reduced across ranks.  The one exchange step is an all-gather of the
owned displacement slabs before the kernels (ghost nodes need u); nothing follows the kernels, and the summation order
(ascending global element id) is the same on every rank, so the sharded matrix is bit-identical to the single-GPU one.

Host logic only (numpy + torch.distributed for the plumbing); every arithmetic step of the path still runs in the CUDA
kernels behind FemContext.  `partition` and `exchange_u` have no GPU dependency and are covered by a world-2 gloo test.
"""
import numpy as np


def partition(n_nodes, conn, world, rank):
    """Node slab [n0, n1) of `rank`, its local mesh and index maps.

    Local nodes keep the global order (sorted global ids), local elements keep ascending global id: neighbour lists, CSR
    column order and the per-entry summation order of the local problem are those of the global one.
    Returns dict(n0, n1, elems, lnodes, lconn, lo, hi): elems = global ids of the local elements, lnodes = global ids of the
    local nodes, lconn = local connectivity (int32), [lo, hi) = local indices of the owned nodes (contiguous)."""
    conn = np.asarray(conn)
    n0, n1 = (rank * n_nodes) // world, ((rank + 1) * n_nodes) // world
    emask = ((conn >= n0) & (conn < n1)).any(axis=1)
    elems = np.flatnonzero(emask)
    lnodes = np.unique(np.concatenate([conn[elems].ravel(), np.arange(n0, n1, dtype=conn.dtype)]))
    lconn = np.searchsorted(lnodes, conn[elems]).astype(np.int32)
    lo, hi = int(np.searchsorted(lnodes, n0)), int(np.searchsorted(lnodes, n1))
    assert hi - lo == n1 - n0
    return dict(n0=n0, n1=n1, elems=elems, lnodes=lnodes, lconn=lconn, lo=lo, hi=hi, world=world, rank=rank, n_nodes=n_nodes)


def exchange_plan(part, device):
    """Index tensors of exchange_u built once per partition (no host work inside the timed step): for every local node its
    row in the padded all-gather buffer [world, width/3, 3]."""
    import torch
    world, n_nodes = part["world"], part["n_nodes"]
    bounds = np.array([((r * n_nodes) // world, ((r + 1) * n_nodes) // world) for r in range(world)], dtype=np.int64)
    width = int((bounds[:, 1] - bounds[:, 0]).max())
    ln = part["lnodes"].astype(np.int64)
    owner = np.searchsorted(bounds[:, 1], ln, side="right")
    gidx = owner * width + (ln - bounds[owner, 0])
    return dict(width=width, gidx=torch.from_numpy(gidx).to(device))


def exchange_u(u_owned, part, group=None, plan=None):
    """The one collective of the sharded path: all-gather of the owned displacement slabs (padded to the largest slab, NCCL
    needs equal counts) -> the displacement of this rank's local nodes, owned and ghost.  u_owned: [3 (n1-n0)] torch tensor
    on the device of the process group's backend; world 1 needs no process group."""
    import torch
    world = part["world"]
    if plan is None:
        plan = exchange_plan(part, u_owned.device)
    width = plan["width"]
    if world == 1:
        full = u_owned.view(-1, 3)
    else:
        import torch.distributed as dist
        send = torch.zeros(3 * width, dtype=u_owned.dtype, device=u_owned.device)
        send[:u_owned.numel()] = u_owned
        recv = torch.empty(world * 3 * width, dtype=u_owned.dtype, device=u_owned.device)
        dist.all_gather_into_tensor(recv, send, group=group)
        full = recv.view(-1, 3)
    return full[plan["gidx"]].reshape(-1).contiguous()


def owned_nnz(row_ptr, part):
    """Number of CSR entries in the rows this rank owns, from the local pattern's row_ptr."""
    return int(row_ptr[3 * part["hi"]]) - int(row_ptr[3 * part["lo"]])


class ShardedFem:
    """fem_setup / fem_build_csr_pattern / fem_assemble of one rank's slab.  Outputs are the owned rows only:
    residual [3 (n1-n0)], csr_vals of rows 3 n0 .. 3 n1 - 1 (contiguous, global column order), hist_out of the local elements."""

    def __init__(self, coords, conn, world, rank, device, fbar=0):
        import torch
        from . import binding as fem
        self.part = partition(coords.shape[0], conn, world, rank)
        p = self.part
        self.device = device
        self.ctx = fem.FemContext(torch.from_numpy(np.ascontiguousarray(coords[p["lnodes"]])).to(device),
                                  torch.from_numpy(p["lconn"]).to(device), fbar=fbar)
        row_ptr, col_idx, _ = self.ctx.build_csr_pattern()
        self.a, self.b = int(row_ptr[3 * p["lo"]].item()), int(row_ptr[3 * p["hi"]].item())
        self.row_ptr = (row_ptr[3 * p["lo"]:3 * p["hi"] + 1] - self.a).contiguous()          # owned rows, rebased
        lcol = col_idx[self.a:self.b].long()
        gl = torch.from_numpy(p["lnodes"].astype(np.int64)).to(device)
        self.col_idx = (3 * gl[lcol // 3] + lcol % 3).to(torch.int32)                        # global column ids
        self.n_elems = p["lconn"].shape[0]

    def assemble(self, u_owned, hist_in_local, mat, group=None, u_local=None):
        """u_owned: this rank's slab of the global displacement; hist_in_local: history of the local elements (global ids
        part['elems']); mat: one record or one per local element.  Returns (residual_owned, csr_vals_owned, hist_out_local).
        u_local (displacement of the local nodes, already exchanged) skips the collective: single-process checks only."""
        p = self.part
        if u_local is None:
            u_local = exchange_u(u_owned, p, group)
        res, vals, hout, _ = self.ctx.assemble(u_local, hist_in_local, mat)
        return res[3 * p["lo"]:3 * p["hi"]], vals[self.a:self.b], hout
