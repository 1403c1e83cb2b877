"""Slab decomposition along k, one process (rank) per GPU: the paper's own parallelisation ("the domain is
decomposed into slabs along one dimension", MPI between ranks), here with torch.distributed (NCCL over NVLink / NVSwitch on
GPUs) as the transport.  SURVEY.md 8(e) / 8(f) NEXT-3.

Per S2O4 step and rank:  dt = all-reduce MIN of the local CFL reductions;  exchange halos of W^n -> stage 1 ->
exchange halos of W* -> stage 2.  A halo is two k-planes of all 80 state fields per side (2 x ni x nj x 640 B: 189 MB per
side at 384^2), packed and unpacked by the library's kernels (cgks_pack_halo / cgks_unpack_halo); the exchange is ~1 % of a
stage at 48 planes per rank, so it is not overlapped with interior work (overlap would cost 12 % recomputed planes).

Everything here is argument marshalling and message choreography; no arithmetic of the method."""
import torch
import torch.distributed as dist

from . import binding

# Message tags, for backends that honour them (gloo, MPI): sender's HIGH planes -> receiver's LOW halo and the reverse.  NCCL's
# point-to-point calls IGNORE tags: messages between one pair of ranks are matched purely by the order in which they are
# posted.  exchange_halos therefore never has two messages in flight in the same direction between the same pair (see there);
# the tags are decoration, not what keeps the ring unambiguous.
UP, DOWN, BOTH = 0, 1, 2


def partition(nk, world):
    """[(k0, nk_owned)] per rank: contiguous slabs of k-planes, sizes differing by at most one, each at least 2 planes."""
    if world < 1 or nk < 2 * world:
        raise ValueError("cannot cut %d planes into %d slabs of at least 2 planes" % (nk, world))
    base, rem = divmod(nk, world)
    out = []; k0 = 0
    for r in range(world):
        cnt = base + (1 if r < rem else 0)
        out.append((k0, cnt)); k0 += cnt
    return out


def neighbours(rank, world):
    """(low, high) ranks of the periodic slab ring."""
    return (rank - 1) % world, (rank + 1) % world


def extended(a, k0, nk_owned, kdim):
    """Planes [k0 - 2, k0 + nk_owned + 2) of a global periodic array (wrapping) along dimension kdim."""
    nk = a.shape[kdim]
    idx = torch.arange(k0 - 2, k0 + nk_owned + 2, device=a.device) % nk
    return a.index_select(kdim, idx).contiguous()


def exchange_halos(sub, rank, world, group=None):
    """Fills both halos of `sub` (anything with halo_buffer / pack_halo / unpack_halo: binding.Solver(slab=...)) from the ring
    neighbours.  The low halo receives the low neighbour's high owned planes, the high halo the high neighbour's low ones."""
    send_lo, send_hi = sub.halo_buffer(), sub.halo_buffer()
    sub.pack_halo(0, send_lo); sub.pack_halo(1, send_hi)
    if world == 1:
        sub.unpack_halo(0, send_hi); sub.unpack_halo(1, send_lo)
        return
    lo, hi = neighbours(rank, world)
    if lo == hi:
        # world == 2: both neighbours are the SAME rank.  Two sends to one peer would be told apart only by tag (ignored by NCCL)
        # or by posting order (an invariant nobody can see at the call site), so both halves travel in ONE message per
        # direction: [low owned planes | high owned planes].  The peer's high planes fill my low halo and the reverse.
        n = send_lo.numel()
        send = torch.cat([send_lo, send_hi]); recv = torch.empty_like(send)
        ops = [dist.P2POp(dist.isend, send, hi, group, BOTH), dist.P2POp(dist.irecv, recv, hi, group, BOTH)]
        for req in dist.batch_isend_irecv(ops):
            req.wait()
        sub.unpack_halo(0, recv[n:]); sub.unpack_halo(1, recv[:n])
        return
    # world >= 3: lo != hi, one message per (peer, direction); nothing to disambiguate, whatever the backend does with tags
    recv_lo, recv_hi = sub.halo_buffer(), sub.halo_buffer()
    ops = [dist.P2POp(dist.isend, send_hi, hi, group, UP), dist.P2POp(dist.isend, send_lo, lo, group, DOWN),
           dist.P2POp(dist.irecv, recv_lo, lo, group, UP), dist.P2POp(dist.irecv, recv_hi, hi, group, DOWN)]
    for req in dist.batch_isend_irecv(ops):
        req.wait()
    sub.unpack_halo(0, recv_lo); sub.unpack_halo(1, recv_hi)


def exchange_halos_local(subs):
    """The same exchange between the sub-domains of ONE process (several contexts on one device): device copies only."""
    bufs = []
    for s in subs:
        lo, hi = s.halo_buffer(), s.halo_buffer()
        s.pack_halo(0, lo); s.pack_halo(1, hi)
        bufs.append((lo, hi))
    w = len(subs)
    for r, s in enumerate(subs):
        lo, hi = neighbours(r, w)
        s.unpack_halo(0, bufs[lo][1]); s.unpack_halo(1, bufs[hi][0])


def global_min(x, device, group=None):
    """Minimum over ranks of a host scalar (the time step: one scalar all-reduce per step)."""
    t = torch.tensor([x], dtype=torch.float64, device=device)
    if dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MIN, group=group)
    return float(t.item())


class SlabSolver:
    """One rank's sub-domain of the global periodic mesh `nodes` (3, nk+1, nj+1, ni+1), with the step choreography."""

    def __init__(self, nodes, params, rank=None, world=None, device=None, budget_bytes=0, group=None):
        self.rank = dist.get_rank(group) if rank is None else rank
        self.world = dist.get_world_size(group) if world is None else world
        self.group = group
        nk = int(nodes.shape[1]) - 1
        self.k0, self.nk_owned = partition(nk, self.world)[self.rank]
        self.sub = binding.Solver(nodes, params, device=device or "cuda:0", budget_bytes=budget_bytes, slab=(self.k0, self.nk_owned))
        self.device = self.sub.device

    def set_state_global(self, Q, G=None, D=None):
        """Global arrays (5, nk, nj, ni) [, (5, 3, ...), (5, 12, ...)]; this rank keeps its slab and halo planes."""
        ext = lambda a, kd: None if a is None else extended(binding._dev(a, self.device), self.k0, self.nk_owned, kd)
        self.sub.set_state(ext(Q, 1), ext(G, 2), ext(D, 2))

    def owned(self, a, kdim):
        return a.narrow(kdim, 2, self.nk_owned)

    def get_state_owned(self):
        Q, G, D = self.sub.get_state()
        return self.owned(Q, 1), self.owned(G, 2), self.owned(D, 2)

    def compute_dt(self, cfl):
        return global_min(self.sub.compute_dt(cfl), self.device, self.group)

    def step(self, dt):
        for stage in (1, 2):
            exchange_halos(self.sub, self.rank, self.world, self.group)
            self.sub.stage(stage, dt)

    def close(self):
        self.sub.close()
