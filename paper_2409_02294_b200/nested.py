"""Nested 3-D mesh levels: who sends what to whom, and when.

The paper runs "the convolution method ... on nested grids", one mesh level per GPU (Fig. 8 :306),
and moves the level-boundary data with one-sided transfers.  Here every step of the arithmetic runs in
the library's kernels (pg3n_* calls, include/polargrav.h, readings M1-M6); this module holds the SCHEDULE only:

    restriction chain   l = D-1 .. 1 :  level l  --(n/2)^3 doubles-->  level l-1        (fine -> coarse)
    solves              every level, independently (own_l, out_l)
    exterior chain      l = 0 .. D-2 :  level l  --(n/2 + 2)^3 doubles-->  level l+1    (coarse -> fine)

`run_schedule` is written against two small protocols, so that the same code drives
  * all levels of one process on ONE GPU, one CUDA stream per level (the "CUDA Streams" the paper leaves unexplored,
    PAPER.md:269): messages are handed over by pointer, ordered by stream events (`LocalLink`);
  * one level per rank / GPU: messages travel by `torch.distributed` send / recv -- NCCL over NVLink on GPUs
    (`DistLink`) -- or ONE-SIDED (`PutLink`, the paper's own model): every level exports its two inboxes by
    CUDA IPC handle, its neighbours open them, and the restriction / packing kernels write their message straight into
    the neighbour's inbox (peer stores over NVLink); all that travels through `torch.distributed` is a one-element
    "it is there" token.  The solves of the levels run concurrently on their own GPUs.
The world-size-2 gloo test drives the same schedule on CPU tensors with stand-in levels (tests/test_multirank_gloo.py).
No arithmetic of the method lives here.
"""
from __future__ import annotations


def message_counts(n: int):
    """(restricted densities upwards, exterior potentials downwards), doubles per level boundary."""
    return (n // 2) ** 3, (n // 2 + 2) ** 3


class LocalLink:
    """All levels in this process.  A message is the sender's buffer itself; `ready(level)` / `wait(level, token)`
    let the level objects order their streams (no-ops for host stand-ins)."""

    def __init__(self):
        self._box = {}

    def send(self, src_level, dst_level, tensor, token=None):
        self._box[(src_level, dst_level)] = (tensor, token)

    def recv(self, src_level, dst_level, like=None):
        return self._box.pop((src_level, dst_level))


class DistLink:
    """One level per rank: level l lives on rank l of `group`.  Blocking send / recv of the message tensors."""

    def __init__(self, dist, group=None):
        self.dist, self.group = dist, group

    def send(self, src_level, dst_level, tensor, token=None):
        if token is not None:
            token.synchronize()                       # the message is complete before it leaves
        self.dist.send(tensor, dst=dst_level, group=self.group)

    def recv(self, src_level, dst_level, like=None):
        self.dist.recv(like, src=src_level, group=self.group)
        return like, None


class PutLink:
    """One level per rank, one-sided: the payload has been PUT into the receiver's inbox by the sender's kernel; send /
    recv move a one-element token that tells the receiver so.  `connect` exchanges the IPC handles once."""

    def __init__(self, dist, group=None, token_device=None):
        import torch
        self.dist, self.group = dist, group
        if token_device is None:       # an NCCL group moves device tensors only, a gloo group host tensors
            token_device = "cuda" if str(dist.get_backend(group)).lower() == "nccl" else "cpu"
        self.tok = torch.zeros(1, dtype=torch.int32, device=token_device)

    def connect(self, level):
        """level: the GpuLevel this rank owns (rank = level index)."""
        pg = level.pg
        mine = {}
        if level.level < level.depth - 1:
            mine["mean"] = pg.pg3n_inbox_export(level.h, pg.PG3N_INBOX_MEAN)[0]
        if level.level > 0:
            mine["halo"] = pg.pg3n_inbox_export(level.h, pg.PG3N_INBOX_HALO)[0]
        everyone = [None] * self.dist.get_world_size(self.group)
        self.dist.all_gather_object(everyone, mine, group=self.group)
        if level.level > 0:                                   # restriction goes into the parent's MEAN inbox
            pg.pg3n_peer_open(level.h, pg.PG3N_INBOX_MEAN, everyone[level.level - 1]["mean"])
        if level.level < level.depth - 1:                     # the exterior potential into the child's HALO inbox
            pg.pg3n_peer_open(level.h, pg.PG3N_INBOX_HALO, everyone[level.level + 1]["halo"])
        level.one_sided = True

    def send(self, src_level, dst_level, tensor, token=None):
        if token is not None:
            token.synchronize()                       # the putting kernel has completed: the message is in the inbox
        self.dist.send(self.tok, dst=dst_level, group=self.group)

    def recv(self, src_level, dst_level, like=None):
        self.dist.recv(self.tok, src=src_level, group=self.group)
        return None, None


def run_schedule(levels, depth, link):
    """levels: {level index: object with restrict() -> (tensor, token), absorb(tensor, token), solve(),
    add_exterior(tensor | None, token), pack_exterior() -> (tensor, token), recv_buffers() -> (mean_like, halo_like)}
    for the levels THIS process owns; link: LocalLink or DistLink.  Every process calls this with the same depth."""
    for l in range(depth - 1, 0, -1):                 # M2: restriction chain, finest first
        if l in levels:
            t, tok = levels[l].restrict()
            link.send(l, l - 1, t, tok)
        if l - 1 in levels:
            t, tok = link.recv(l, l - 1, levels[l - 1].recv_buffers()[0])
            levels[l - 1].absorb(t, tok)
    for l in sorted(levels):                          # M3: independent solves
        levels[l].solve()
    for l in range(depth):                            # M4-M6: exterior chain, coarsest first
        if l in levels:
            if l == 0:
                levels[l].add_exterior(None, None)
            else:
                t, tok = link.recv(l - 1, l, levels[l].recv_buffers()[1])
                levels[l].add_exterior(t, tok)
            if l < depth - 1:
                t, tok = levels[l].pack_exterior()
                link.send(l, l + 1, t, tok)


class GpuLevel:
    """One pg3n_level on its own CUDA stream, with its two outgoing and two incoming message buffers (torch tensors)."""

    def __init__(self, n, box0, level, depth, device):
        import torch
        from . import binding as pg
        self.pg, self.torch = pg, torch
        self.n, self.level, self.depth, self.device = n, level, depth, device
        with torch.cuda.device(device):
            self.stream = torch.cuda.Stream()
            self.h = pg.pg3n_create(n, box0, level, depth, device, self.stream.cuda_stream)
            n_mean, n_halo = message_counts(n)
            mk = lambda c: torch.empty(c, dtype=torch.float64, device=f"cuda:{device}")
            self.mean_out, self.halo_out, self.mean_in, self.halo_in = mk(n_mean), mk(n_halo), mk(n_mean), mk(n_halo)
        self.one_sided = False        # PutLink.connect: messages are written into / read from the inboxes of the library

    def recv_buffers(self):
        return self.mean_in, self.halo_in

    def _token(self):
        ev = self.torch.cuda.Event()
        ev.record(self.stream)
        return ev

    def _after(self, token):
        if token is not None:
            self.stream.wait_event(token)
        else:
            self.stream.wait_stream(self.torch.cuda.current_stream(self.device))    # a message received by NCCL

    def set_density(self, rho):
        self.stream.wait_stream(self.torch.cuda.current_stream(self.device))
        self.pg.pg3n_set_density(self.h, rho, self.pg.PG_MEM_DEVICE)

    def restrict(self):
        out = None if self.one_sided else self.mean_out
        self.pg.pg3n_restrict(self.h, out)
        return out, self._token()

    def absorb(self, t, token):
        if t is not None or self.one_sided:
            self._after(token)                # one-sided: behind the token's receive (stream-ordered with nccl tokens)
        self.pg.pg3n_absorb(self.h, t)        # None: this level's MEAN inbox (the token has been received: it is there)

    def solve(self):
        self.pg.pg3n_solve(self.h)

    def add_exterior(self, t, token):
        if t is not None or (self.one_sided and self.level > 0):
            self._after(token)
        self.pg.pg3n_add_exterior(self.h, t)  # None: level 0, or (one-sided) this level's HALO inbox

    def pack_exterior(self):
        out = None if self.one_sided else self.halo_out
        self.pg.pg3n_pack_exterior(self.h, out)
        return out, self._token()

    def potential(self, out):
        self.pg.pg3n_potential(self.h, out, self.pg.PG_MEM_DEVICE)

    def synchronize(self):
        self.pg.pg3n_synchronize(self.h)

    def close(self):
        if self.h is not None:
            self.pg.pg3n_destroy(self.h)
            self.h = None


class NestedPotential:
    """depth levels of n^3 cells.  world_size 1: all levels on `device`, one stream each.  world_size == depth
    (torch.distributed initialised, backend nccl): this rank owns level `rank` on its own GPU."""

    def __init__(self, n, box0, depth, device=0, dist=None, group=None, link="put", token_device=None):
        """link (world_size > 1 only): "put" = one-sided puts into the neighbours' inboxes (PutLink), "sendrecv" =
        payloads by torch.distributed send / recv (DistLink; needs a backend that moves device tensors, i.e. nccl)."""
        self.n, self.box0, self.depth = n, box0, depth
        world = dist.get_world_size(group) if dist is not None else 1
        if world == 1:
            self.owned = list(range(depth))
            self.link = LocalLink()
        else:
            if world != depth:
                raise ValueError(f"one level per rank: world size {world} != depth {depth}")
            self.owned = [dist.get_rank(group)]
            if token_device is None and str(dist.get_backend(group)).lower() == "nccl":
                token_device = f"cuda:{device}"       # the level's own GPU; PutLink picks "cpu" for gloo
            self.link = PutLink(dist, group, token_device) if link == "put" else DistLink(dist, group)
        self.levels = {l: GpuLevel(n, box0, l, depth, device) for l in self.owned}
        if isinstance(self.link, PutLink):
            self.link.connect(self.levels[self.owned[0]])

    def solve(self, rhos, outs):
        """rhos / outs: {level: device tensor [n][n][n]} for the owned levels.  Enqueues; call synchronize()."""
        for l in self.owned:
            self.levels[l].set_density(rhos[l])
        run_schedule(self.levels, self.depth, self.link)
        for l in self.owned:
            self.levels[l].potential(outs[l])

    def synchronize(self):
        for l in self.owned:
            self.levels[l].synchronize()

    def launches(self):
        return sum(self.levels[l].pg.pg3n_launch_count(self.levels[l].h) for l in self.owned)

    def close(self):
        if isinstance(self.link, PutLink):
            # an exported inbox may not be freed while a neighbour still has it open: everybody lets go first
            for l in self.owned:
                lev = self.levels[l]
                if lev.h is not None:
                    if lev.level > 0:
                        lev.pg.pg3n_peer_set(lev.h, lev.pg.PG3N_INBOX_MEAN, None)
                    if lev.level < lev.depth - 1:
                        lev.pg.pg3n_peer_set(lev.h, lev.pg.PG3N_INBOX_HALO, None)
            self.link.dist.barrier(group=self.link.group)
        for l in self.owned:
            self.levels[l].close()
