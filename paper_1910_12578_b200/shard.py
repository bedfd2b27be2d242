"""The box lattice sharded over ranks ("MPI distribute the AMR grids across nodes").

One process per GPU.  The global lattice of boxes is cut into equal bricks, one per rank; within one <A(U)>
evaluation the only data that crosses ranks is the 4-deep ghost shell of boxes on a brick surface, plus one scalar
MIN for dt.  Everything here is plumbing: the ghost map, the packing and the unpacking run in the library
(csrc/exchange.cu: cst_set_sublattice, cst_exchange_pack / _unpack); the messages travel through torch.distributed
point-to-point calls (NCCL send/recv over NVLink on GPUs, gloo in the CPU tests).
"""
import numpy as np


def brick_partition(global_nb, world):
    """part[0] x part[1] x part[2] = world ranks, each global_nb[d] divisible by part[d]; cuts the longest
    remaining brick side first (on ties the direction cut least so far), which keeps the bricks as cubic as the
    lattice allows: configs[4]'s 16 x 8 x 4 lattice gives (2,1,1), (2,2,1), (4,2,1) for 2, 4, 8 ranks."""
    part, lb, w = [1, 1, 1], [int(x) for x in global_nb], int(world)
    while w > 1:
        f = next(p for p in (2, 3, 5, 7, w) if w % p == 0)
        cand = [d for d in range(3) if lb[d] % f == 0]
        if not cand:
            raise ValueError(f"cannot cut a {tuple(global_nb)} lattice into {world} equal bricks")
        d = max(cand, key=lambda d: (lb[d], -part[d], -d))
        part[d] *= f
        lb[d] //= f
        w //= f
    return tuple(part)


def rank_coords(part, rank):
    return rank % part[0], (rank // part[0]) % part[1], rank // (part[0] * part[1])


def local_config(cfg_global, part):
    """Config of one rank's brick: same zones per box, widths, BCs (of the GLOBAL domain), brick lattice."""
    c = dict(cfg_global)
    for k, d in (("nbx", 0), ("nby", 1), ("nbz", 2)):
        if cfg_global[k] % part[d]:
            raise ValueError("lattice not divisible by the partition")
        c[k] = cfg_global[k] // part[d]
    return c


def local_boxes(cfg_global, part, rank):
    """Global box indices of the rank's brick, in the brick's local box order."""
    lb = [cfg_global[k] // part[d] for k, d in (("nbx", 0), ("nby", 1), ("nbz", 2))]
    p = rank_coords(part, rank)
    out = []
    for bk in range(lb[2]):
        for bj in range(lb[1]):
            for bi in range(lb[0]):
                g = (p[0] * lb[0] + bi, p[1] * lb[1] + bj, p[2] * lb[2] + bk)
                out.append(g[0] + cfg_global["nbx"] * (g[1] + cfg_global["nby"] * g[2]))
    return np.array(out)


class GhostExchange:
    """Ghost fill of a sharded lattice.  Two transports:

    mode="sendrecv" (default): local fill + cst_exchange_pack + one torch.distributed point-to-point message per peer
        + cst_exchange_unpack (NCCL send/recv on GPUs, gloo in the CPU tests);
    mode="p2p": local fill + cst_exchange_push -- ONE kernel that stores every zone the peers' shells read from this
        brick straight into the peers' arrays through peer-mapped pointers (CUDA IPC over NVLink / NVSwitch), no staging
        buffers, no communication library on the data path; two barriers separate the pushes from the peers' reads.
        Every state array that is ghost-filled must be registered once (register(U)): its IPC handle goes to the peers.

    ctx: binding.Context of the rank's brick (local_config) -- set_sublattice is called here.
    alloc(n_doubles) -> a float64 buffer on the device of U (torch tensor)."""

    def __init__(self, ctx, cfg_global, part, rank, alloc, mode="sendrecv"):
        self.ctx, self.rank, self.mode = ctx, rank, mode
        ctx.set_sublattice((cfg_global["nbx"], cfg_global["nby"], cfg_global["nbz"]), part, rank)
        self.info = ctx.exchange_info()
        ns = sum(i[2] for i in self.info)
        nr = sum(i[4] for i in self.info)
        self.bytes_per_fill = 8 * (ns + nr)
        self._peer_ptrs = {}                    # data_ptr of a registered U -> the peers' mapped addresses
        self._mapped = []
        if mode == "sendrecv":
            self.sendbuf, self.recvbuf = alloc(max(ns, 1)), alloc(max(nr, 1))
        elif mode != "p2p":
            raise ValueError("mode must be 'sendrecv' or 'p2p'")

    def register(self, U):
        """p2p: make U reachable by the peers and map their corresponding arrays (collective: every rank calls it with
        its own array, in the same order)."""
        import torch.distributed as dist
        from . import binding
        handle, off = binding.ipc_export(U)
        everyone = [None] * dist.get_world_size()
        dist.all_gather_object(everyone, (handle, off))
        ptrs = []
        for peer, *_ in self.info:
            addr = binding.ipc_import(*everyone[peer])
            self._mapped.append(addr - everyone[peer][1])
            ptrs.append(addr)
        self._peer_ptrs[U.data_ptr()] = ptrs

    def close(self):
        from . import binding
        for base in self._mapped:
            binding.ipc_close(base)
        self._mapped, self._peer_ptrs = [], {}

    def fill_ghosts(self, U, stream=None):
        """Complete ghost fill of the local boxes of U (in place)."""
        import torch.distributed as dist
        if self.mode == "p2p" and self.info:
            import torch
            dist.barrier()                      # the peers have finished reading the shells this push overwrites
            self.ctx.fill_ghosts(U, stream)
            self.ctx.exchange_push(U, self._peer_ptrs[U.data_ptr()], stream)
            torch.cuda.synchronize()            # my stores have landed ...
            dist.barrier()                      # ... and so have everyone else's
            return
        self.ctx.fill_ghosts(U, stream)
        if not self.info:
            return
        self.ctx.exchange_pack(U, self.sendbuf, stream)
        ops = []
        for peer, so, sl, ro, rl in self.info:
            if rl:
                ops.append(dist.P2POp(dist.irecv, self.recvbuf[ro:ro + rl], peer))
            if sl:
                ops.append(dist.P2POp(dist.isend, self.sendbuf[so:so + sl], peer))
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        self.ctx.exchange_unpack(U, self.recvbuf, stream)


def allreduce_min(x, device):
    """MIN of a host scalar over the ranks (the time step)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return float(t.item())
