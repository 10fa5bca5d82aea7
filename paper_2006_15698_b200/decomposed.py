"""Block decomposition of one mesh over several contexts / GPUs.

The paper's coarse-grain parallelism is an MPI mesh decomposition with one exchange of face data per Runge-Kutta
stage.  Here: one process per GPU, `torch.distributed` (NCCL over NVLink / NVSwitch) for the plumbing, and the
library's face export / import (dg_halo_export, dg_set_halo, dg_rk_stage in include/dg_b200.h) for the data: a rank's
context treats the faces it shares with other ranks as DG_BC_HALO faces, exports the traces of its own boundary
elements after every stage and receives the neighbours' straight into the buffers its kernels read.  All arithmetic
stays in the CUDA kernels; this module is argument marshalling and message plumbing only.

`Decomposition` is pure host logic (no torch, no GPU): who owns which elements, who is whose neighbour across which
face, in which order messages are posted.  `DistributedDG` is one rank's part of the mesh.  The exchange itself is a
callable, so that the tests can run several ranks' contexts inside one process on one GPU (copies instead of messages).
"""
PERIODIC, WALL, FARFIELD, HALO = 0, 1, 2, 3
FACES = ("x-", "x+", "y-", "y+", "z-", "z+")


def _split(n, parts):
    """Element ranges of `parts` contiguous pieces of 0..n, sizes differing by at most one."""
    base, extra = divmod(n, parts)
    out, lo = [], 0
    for i in range(parts):
        hi = lo + base + (1 if i < extra else 0)
        out.append((lo, hi))
        lo = hi
    return out


class Decomposition:
    """procs = (px, py, pz) ranks along x, y, z; rank = cx + px * (cy + py * cz).  bc = the GLOBAL domain's conditions
    (x-, x+, y-, y+, z-, z+), values as in include/dg_b200.h."""

    def __init__(self, n, procs, bc=(PERIODIC,) * 6):
        self.n = tuple(int(v) for v in n)
        self.procs = tuple(int(v) for v in procs)
        self.bc = tuple(int(v) for v in bc)
        if any(p < 1 for p in self.procs) or any(p > m for p, m in zip(self.procs, self.n)):
            raise ValueError("every rank needs at least one element along every axis")
        for a in range(3):
            if (self.bc[2 * a] == PERIODIC) != (self.bc[2 * a + 1] == PERIODIC):
                raise ValueError("an axis is periodic on both of its faces or on neither")
        self.size = self.procs[0] * self.procs[1] * self.procs[2]
        self.ranges = [_split(self.n[a], self.procs[a]) for a in range(3)]

    def coords(self, rank):
        px, py, _ = self.procs
        return (rank % px, (rank // px) % py, rank // (px * py))

    def rank_of(self, c):
        px, py, _ = self.procs
        return c[0] + px * (c[1] + py * c[2])

    def local_box(self, rank):
        """((x0, x1), (y0, y1), (z0, z1)): the rank's element ranges in the global mesh."""
        c = self.coords(rank)
        return tuple(self.ranges[a][c[a]] for a in range(3))

    def local_n(self, rank):
        return tuple(hi - lo for lo, hi in self.local_box(rank))

    def neighbour(self, rank, face):
        """Rank owning the elements beyond `face` of `rank`, or None on a non-periodic domain face.  With one rank
        along a periodic axis the neighbour is the rank itself (the context then simply stays periodic there)."""
        a, side = face // 2, face % 2
        c = list(self.coords(rank))
        c[a] += 1 if side else -1
        if c[a] < 0 or c[a] >= self.procs[a]:
            if self.bc[face] != PERIODIC:
                return None
            c[a] %= self.procs[a]
        return self.rank_of(c)

    def local_bc(self, rank):
        """Boundary conditions of the rank's context: HALO where another rank is the neighbour."""
        out = []
        for f in range(6):
            nb = self.neighbour(rank, f)
            if nb is None:
                out.append(self.bc[f])
            elif nb == rank:
                out.append(PERIODIC)
            else:
                out.append(HALO)
        return tuple(out)

    def sends(self, rank):
        """[(face, neighbour)] in the order this rank posts its sends: face order.  The export of face f feeds the
        neighbour's face f ^ 1."""
        return [(f, nb) for f in range(6) for nb in [self.neighbour(rank, f)] if nb is not None and nb != rank]

    def recvs(self, rank):
        """[(my face, neighbour)] in the order this rank posts its receives: for every peer, the order in which THAT
        peer posts its sends to me (point-to-point messages between two ranks match in posting order)."""
        out = []
        for peer in range(self.size):
            if peer == rank:
                continue
            for f, nb in self.sends(peer):
                if nb == rank:
                    out.append((f ^ 1, peer))
        return out


def choose_variant(dec, p, shapes):
    """One column shape for ALL ranks (neighbours must agree on the face-trace layout): the first compiled variant
    (they are listed fastest first) that pads no rank's local mesh by 4 % or more, else the one that pads least.
    shapes = [(bx, by)] of the compiled variants of degree p."""
    worst = []
    for bx, by in shapes:
        w = 0.0
        for r in range(dec.size):
            nx, ny, _ = dec.local_n(r)
            padded = (-(-nx // bx) * bx) * (-(-ny // by) * by)
            w = max(w, padded / float(nx * ny) - 1.0)
        worst.append(w)
    for v, w in enumerate(worst):
        if w < 0.04:
            return v
    return min(range(len(shapes)), key=lambda v: worst[v])


def variant_shapes(p):
    """(bx, by) of every stage-kernel variant compiled for degree p."""
    from .binding import DG, load_library
    out = []
    for v in range(load_library().dg_variant_count(p)):
        probe = DG(8, 8, 8, p, bind=False, variant=v)
        info = probe.kernel_info()
        out.append((info["bx"], info["by"]))
        probe.close()
    return out


def exchange_torch_distributed(dist):
    """Face exchange over torch.distributed point-to-point operations (NCCL: GPU buffers over NVLink)."""
    def run(rank, sends, recvs):
        ops = [dist.P2POp(dist.isend, buf, peer, tag=face) for face, peer, buf in sends]
        ops += [dist.P2POp(dist.irecv, buf, peer, tag=face ^ 1) for face, peer, buf in recvs]
        if ops:
            for req in dist.batch_isend_irecv(ops):
                req.wait()
    return run


class DistributedDG:
    """One rank's block of a decomposed mesh.  `q` arrays are the rank's LOCAL canonical arrays
    (nz_l, ny_l, nx_l, N, N, N, 5); `exchange(rank, sends, recvs)` moves [(face, peer, tensor)] lists (default:
    torch.distributed); `reduce_max(x)` returns the maximum of a float over all ranks (default: all_reduce)."""

    def __init__(self, n, p, gamma, extent, procs, rank, bc=(PERIODIC,) * 6, q_inf=None, device="cuda:0", exchange=None,
                 reduce_max=None, variant=None, push=False):
        import torch
        from .binding import DG
        self.dec = Decomposition(n, procs, bc)
        self.rank, self.p = int(rank), int(p)
        self.box = self.dec.local_box(self.rank)
        nl = self.dec.local_n(self.rank)
        ext_l = tuple(extent[a] * nl[a] / float(self.dec.n[a]) for a in range(3))
        if variant is None:
            variant = choose_variant(self.dec, p, variant_shapes(p))
        # the element sizes are those of the GLOBAL mesh, the same doubles on every rank
        self.dg = DG(*nl, p, gamma, ext_l, device=device, variant=variant,
                     spacing=tuple(extent[a] / float(self.dec.n[a]) for a in range(3)))
        self.local_bc = self.dec.local_bc(self.rank)
        self.dg.set_boundary(self.local_bc, q_inf)
        dev = self.dg.device
        self._send = [(f, nb, torch.empty(self.dg.halo_len(f), dtype=torch.float64, device=dev)) for f, nb in self.dec.sends(self.rank)]
        self._recv = [(f, nb, torch.empty(self.dg.halo_len(f), dtype=torch.float64, device=dev)) for f, nb in self.dec.recvs(self.rank)]
        self.push = bool(push)
        if self.push:
            # push mode (dg_set_halo_pair / dg_set_halo_push): every halo face reads a PAIR of buffers alternately; the
            # neighbour's stage kernel stores its traces straight into them.  connect_push() wires the two sides up.
            self.pairs = {f: (buf, torch.empty_like(buf)) for f, _, buf in self._recv}
            for f, (b0, b1) in self.pairs.items():
                self.dg.set_halo_pair(f, b0, b1)
        else:
            for f, _, buf in self._recv:
                self.dg.set_halo(f, buf)
        self._dist = None
        if self.push and exchange is None:
            import torch.distributed as dist
            self._dist = dist
            self._wire_push_over_ipc(dist)
        if exchange is None or reduce_max is None:
            import torch.distributed as dist
            if exchange is None:
                exchange = exchange_torch_distributed(dist)
            if reduce_max is None:
                def reduce_max(x):
                    # (a CPU tensor where the process group has no CUDA backend, e.g. gloo in the tests)
                    on_gpu = dist.get_backend() == "nccl"
                    t = torch.tensor([x], dtype=torch.float64, device=dev if on_gpu else "cpu")
                    dist.all_reduce(t, op=dist.ReduceOp.MAX)
                    return float(t.item())
        self._exchange, self._reduce_max = exchange, reduce_max

    def connect_push(self, face, peer0, peer1):
        """Push mode: this rank's stage kernels store the traces of face `face` into the neighbour's pair for its face
        `face ^ 1` (tensors of this process, or raw addresses of peer-mapped memory opened through CUDA IPC)."""
        self._push_targets = getattr(self, "_push_targets", {})
        self._push_targets[face] = (peer0, peer1)
        self.dg.set_halo_push(face, peer0, peer1)

    def _wire_push_over_ipc(self, dist):
        """One process per rank: every rank publishes CUDA IPC handles of its halo-buffer pairs (torch's own tensor
        sharing), opens its neighbours' and hands them to the library as push targets.  The mapped buffers may live on
        another GPU: the stage kernel's stores then go over NVLink (dg_set_halo_push enables peer access from this rank's
        device to the buffers' device; never run on more than one GPU so far)."""
        from torch.multiprocessing.reductions import reduce_tensor
        mine = {f: (reduce_tensor(b0), reduce_tensor(b1)) for f, (b0, b1) in self.pairs.items()}
        everyone = [None] * dist.get_world_size()
        dist.all_gather_object(everyone, mine)
        self._peer_tensors = {}
        for f, nb in self.dec.sends(self.rank):
            (fn0, args0), (fn1, args1) = everyone[nb][f ^ 1]
            t0, t1 = fn0(*args0), fn1(*args1)
            self._peer_tensors[f] = (t0, t1)             # keeps the mapping alive
            self.connect_push(f, t0.data_ptr(), t1.data_ptr())
        dist.barrier()

    def _stage_barrier(self):
        """Push mode between processes: every rank has finished its stage (its stores have landed in the neighbours'
        buffers) before anyone starts the next one."""
        self.dg.stream.synchronize()
        self._dist.barrier()

    # the two halves of an exchange are separate so that a single process can drive several ranks (tests)
    def export_faces(self):
        for f, _, buf in self._send:
            self.dg.halo_export(f, buf)
        return self._send

    def exchange(self):
        if not self._send and not self._recv:
            return
        self.export_faces()
        self.dg.stream.synchronize()                 # the messages read buffers written on the library's stream
        self._exchange(self.rank, self._send, self._recv)

    def set_state(self, q_local):
        self.dg.set_state(q_local)
        if self.push and self._dist is not None:
            for f, _ in self.dec.sends(self.rank):     # the initial traces go to the neighbours' buffer 0 (parity 0)
                self.dg._check(self.dg.lib.dg_halo_export(self.dg._h, f, self._push_targets[f][0]))
            self._stage_barrier()
        else:
            self.exchange()
        return self

    def residual(self, out=None):
        return self.dg.residual(out)

    def max_wavespeed(self):
        return self._reduce_max(self.dg.max_wavespeed())

    def rk_step(self, dt, nsteps=1):
        for _ in range(int(nsteps)):
            for stage in range(5):
                self.dg.rk_stage(dt, stage)
                if self.push and self._dist is not None:
                    self._stage_barrier()              # the stage kernel itself has delivered the faces
                else:
                    self.exchange()
        return self

    def rk_step_cfl(self, cfl, nsteps=1):
        """nsteps steps, each with the CFL time step of reading R10 from the maximum wavespeed over ALL ranks; the
        library forms dt (dg_cfl_dt; every block was given the global element sizes).  Returns the time advanced."""
        t = 0.0
        for _ in range(int(nsteps)):
            dt = self.dg.cfl_dt(cfl, self.max_wavespeed())
            self.rk_step(dt, 1)
            t += dt
        return t

    def get_state(self, out=None):
        return self.dg.get_state(out)

    def close(self):
        self.dg.close()


# ------------------------------------------------------------------------------------------------------------------
# several ranks' contexts inside ONE process on one GPU (tests; no messages, no kernels waiting on one another:
# every rank's stage is an ordinary launch, the faces move by device copies in between)
# ------------------------------------------------------------------------------------------------------------------
def exchange_in_process(ranks):
    """ranks: list of DistributedDG indexed by rank, all in this process."""
    exports = {}
    for r in ranks:
        for f, _, buf in r.export_faces():
            exports[(r.rank, f)] = buf
    for r in ranks:
        for f, peer, buf in r._recv:
            buf.copy_(exports[(peer, f ^ 1)])


def make_in_process(n, p, gamma, extent, procs, bc=(PERIODIC,) * 6, q_inf=None, device="cuda:0", variant=None):
    dec = Decomposition(n, procs, bc)
    if variant is None:
        variant = choose_variant(dec, p, variant_shapes(p))
    nothing = lambda rank, sends, recvs: None
    return [DistributedDG(n, p, gamma, extent, procs, r, bc, q_inf, device, exchange=nothing, reduce_max=lambda x: x,
                          variant=variant) for r in range(dec.size)]


def set_state_in_process(ranks, q_global):
    """q_global: the global canonical array (nz, ny, nx, N, N, N, 5); every rank takes its block."""
    import numpy as np
    for r in ranks:
        (x0, x1), (y0, y1), (z0, z1) = r.box
        r.dg.set_state(np.ascontiguousarray(q_global[z0:z1, y0:y1, x0:x1]))
    exchange_in_process(ranks)


def rk_step_in_process(ranks, dt, nsteps=1):
    for _ in range(int(nsteps)):
        for stage in range(5):
            for r in ranks:
                r.dg.rk_stage(dt, stage)
            exchange_in_process(ranks)


def rk_step_cfl_in_process(ranks, cfl, nsteps=1):
    """The CFL-stepped run of all ranks: the wavespeed is the maximum over the ranks, the library forms dt (dg_cfl_dt)."""
    t = 0.0
    for _ in range(int(nsteps)):
        dt = ranks[0].dg.cfl_dt(cfl, max(r.dg.max_wavespeed() for r in ranks))
        rk_step_in_process(ranks, dt, 1)
        t += dt
    return t


def gather_in_process(ranks, what="state"):
    """Global canonical array assembled from the ranks' blocks (what = "state" or "residual")."""
    import numpy as np
    dec = ranks[0].dec
    N = ranks[0].p + 1
    out = np.empty((dec.n[2], dec.n[1], dec.n[0], N, N, N, 5))
    for r in ranks:
        (x0, x1), (y0, y1), (z0, z1) = r.box
        out[z0:z1, y0:y1, x0:x1] = r.dg.get_state() if what == "state" else r.dg.residual()
    return out


# ------------------------------------------------------------------------------------------------------------------
# push mode (dg_set_halo_pair / dg_set_halo_push): the stage kernels store the boundary traces straight into the
# neighbour contexts' halo buffers, no export kernel, no message.  Between processes the buffers are opened in the
# neighbour's address space with CUDA IPC and the stores travel over NVLink; the only communication left is the
# ordering "every rank has finished stage s before anyone starts stage s + 1" (a barrier) -- written here for contexts
# of ONE process, where one stream provides that ordering.
# ------------------------------------------------------------------------------------------------------------------
def make_in_process_push(n, p, gamma, extent, procs, bc=(PERIODIC,) * 6, q_inf=None, device="cuda:0", variant=None):
    dec = Decomposition(n, procs, bc)
    if variant is None:
        variant = choose_variant(dec, p, variant_shapes(p))
    nothing = lambda rank, sends, recvs: None
    ranks = [DistributedDG(n, p, gamma, extent, procs, r, bc, q_inf, device, exchange=nothing, reduce_max=lambda x: x,
                           variant=variant, push=True) for r in range(dec.size)]
    for r in ranks:
        for f, nb in dec.sends(r.rank):
            r.connect_push(f, *ranks[nb].pairs[f ^ 1])
    return ranks


def set_state_in_process_push(ranks, q_global):
    """Every rank takes its block; the traces of the initial state go to the neighbours' buffer 0 (parity 0)."""
    import numpy as np
    for r in ranks:
        (x0, x1), (y0, y1), (z0, z1) = r.box
        r.dg.set_state(np.ascontiguousarray(q_global[z0:z1, y0:y1, x0:x1]))
    for r in ranks:
        for f, nb in r.dec.sends(r.rank):
            r.dg.halo_export(f, ranks[nb].pairs[f ^ 1][0])


def rk_step_in_process_push(ranks, dt, nsteps=1):
    """No exchange step at all: the stage kernels have already put the traces where the neighbours read them."""
    for _ in range(int(nsteps)):
        for stage in range(5):
            for r in ranks:
                r.dg.rk_stage(dt, stage)
