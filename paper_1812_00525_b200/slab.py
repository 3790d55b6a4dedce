"""NEXT-4: Z-slab domain decomposition of the CLTx hot path ("four-layer grids are used for message
passing between every two neighboring blocks", L250-256, L337).

The paper splits its domain in R and exchanges device pointers through MPI.  Here the global grid is cut into slabs
along Z (R is the contiguous axis of the layout, so a ghost block is whole rows): rank r owns the interior rows
[a_r, b_r) of the global grid and runs an ordinary libclt context on the rows [z0, z0 + nZ_local) = its owned rows
plus GHOST = 4 rows per cut (or the two frozen boundary rows at the outer edges).  The kernels are unchanged: they
never write the two outer rows of a context, they recompute rows 2-3 next to a cut from the ghost data (those values
are discarded), and after every RK stage all 4 ghost rows of the stage's output buffer hold the neighbour's freshly
computed owned rows: slabs of one process get them written by the neighbour's stage kernel itself (clt_link_rows: peer
stores from the RK4 epilogue), slabs of different processes by four exchanges of 4 rows x 8 fields per cut and step.

Host logic only (argument marshalling, partition arithmetic, exchange order); every number is computed by the CUDA
kernels behind ``clt.Clt``.  Two drivers over the same code:
  * in-process: several slabs in one process (one or several GPUs), ghost rows handed over as device tensors;
  * torch.distributed: one slab per process, ghost rows by batched isend/irecv (NCCL over NVLink on GPUs).
Never imports ``oracle``.
"""
from __future__ import annotations

import numpy as np

GHOST = 4
STAGE_BUFFER = {1: 1, 2: 2, 3: 1, 4: 0}      # buffer (include/clt.h: 0 = U^n, 1 = U_a, 2 = U_b) written by each stage


def partition(nZ: int, world: int):
    """Owned interior rows [a_r, b_r) of the global interior rows 2 .. nZ-3, as equal as possible."""
    interior = nZ - 4
    if world < 1 or interior < GHOST * world:
        raise ValueError(f"cannot cut {interior} interior rows into {world} slabs of at least {GHOST} rows")
    base, extra = divmod(interior, world)
    out, a = [], 2
    for r in range(world):
        b = a + base + (1 if r < extra else 0)
        out.append((a, b))
        a = b
    return out


class Extent:
    """Row bookkeeping of one slab.  Global row g of rank r is local row g - z0."""

    def __init__(self, nZ: int, world: int, rank: int):
        parts = partition(nZ, world)
        self.nZ, self.world, self.rank = nZ, world, rank
        self.a, self.b = parts[rank]
        self.z0 = 0 if rank == 0 else self.a - GHOST
        self.z1 = nZ if rank == world - 1 else self.b + GHOST          # one past the last local row (global index)
        self.nZ_local = self.z1 - self.z0
        self.lower = rank - 1 if rank > 0 else None
        self.upper = rank + 1 if rank < world - 1 else None

    # local row ranges (first row, count) of the four ghost transfers
    def send_down(self):      # my first GHOST owned rows -> upper ghost rows of rank-1
        return self.a - self.z0, GHOST

    def send_up(self):        # my last GHOST owned rows -> lower ghost rows of rank+1
        return self.b - GHOST - self.z0, GHOST

    def recv_from_lower(self):
        return 0, GHOST

    def recv_from_upper(self):
        return self.nZ_local - GHOST, GHOST

    def owned_local(self):
        return self.a - self.z0, self.b - 1 - self.z0

    def deep_local(self):
        """Rows of max |div_c B|: the global deep interior 4 .. nZ-5 restricted to the owned rows."""
        lo, hi = max(self.a, 4), min(self.b - 1, self.nZ - 5)
        if lo > hi:
            return 2, 1      # empty
        return lo - self.z0, hi - self.z0


def exchange(backends, extents, buffer, dist=None, make_buffer=None):
    """Overwrites the ghost rows of `buffer` in every slab with the neighbours' owned rows.

    backends: the local slab objects (each with get_rows(buffer, k0, n, out) / set_rows(buffer, k0, n, src));
    extents: their Extent.  In-process (dist is None) `backends` holds all ranks in rank order.  With torch.distributed
    it holds this process's one slab and the rows travel by batch_isend_irecv.  make_buffer(n) allocates a dense
    [8][nphi][n][nR] float64 tensor on the transfer device."""
    if dist is None:
        for lo, hi, elo, ehi in zip(backends[:-1], backends[1:], extents[:-1], extents[1:]):
            if hasattr(lo, "push_rows"):
                # one kernel per direction, straight from the owner's buffer into the neighbour's ghost rows, stream-ordered
                lo.push_rows(buffer, *elo.send_up(), hi, ehi.recv_from_lower()[0])
                hi.push_rows(buffer, *ehi.send_down(), lo, elo.recv_from_upper()[0])
                continue
            up = make_buffer(lo, GHOST)
            lo.get_rows(buffer, *elo.send_up(), up)
            down = make_buffer(hi, GHOST)
            hi.get_rows(buffer, *ehi.send_down(), down)
            hi.set_rows(buffer, *ehi.recv_from_lower(), up.to(down.device) if hasattr(up, "to") else up)
            lo.set_rows(buffer, *elo.recv_from_upper(), down.to(up.device) if hasattr(down, "to") else down)
        return
    (be,), (ex,) = backends, extents
    ops, landing = [], []
    for peer, send_rows, recv_rows in ((ex.lower, ex.send_down(), ex.recv_from_lower()),
                                       (ex.upper, ex.send_up(), ex.recv_from_upper())):
        if peer is None:
            continue
        out = make_buffer(be, GHOST)
        be.get_rows(buffer, *send_rows, out)
        inc = make_buffer(be, GHOST)
        ops.append(dist.P2POp(dist.isend, out, peer))
        ops.append(dist.P2POp(dist.irecv, inc, peer))
        landing.append((recv_rows, inc, out))
    if ops:
        for req in dist.batch_isend_irecv(ops):
            req.wait()
    for recv_rows, inc, _keep in landing:
        be.set_rows(buffer, *recv_rows, inc)


class Slab:
    """One sub-domain: a libclt context on the rows of `Extent`, built from the GLOBAL arrays."""

    def __init__(self, cfg, dt, U0, U, rank, world, device="cuda:0", d_i=0.0, phi_scheme=0, stream=None):
        import torch
        from . import clt
        self.ext = ex = Extent(cfg.nZ, world, rank)
        dZ = (cfg.Zmax - cfg.Zmin) / (cfg.nZ - 1)
        Zmin = cfg.Zmin + ex.z0 * dZ
        Zmax = cfg.Zmin + (ex.z1 - 1) * dZ
        self.g = clt.Clt(cfg.nR, cfg.nphi, ex.nZ_local, cfg.Rmin, cfg.Rmax, Zmin, Zmax, cfg.phi_extent, cfg.gamma, cfg.eta,
                         cfg.nu, cfg.D, cfg.kappa, dt, cfg.cfl, d_i=d_i, device=device, stream=stream)
        self.g.set_z_spacing(dZ)      # the global spacing itself, not (Zmax - Zmin)/(nZ_local - 1): slabs == undivided run, bit for bit
        if phi_scheme:
            self.g.set_phi_scheme(phi_scheme)
        self.device = torch.device(device)
        self.row_shape = (8, cfg.nphi, GHOST, cfg.nR)
        if U0 is not None:
            self.g.set_equilibrium(np.ascontiguousarray(U0[:, ex.z0:ex.z1]))
        self.g.set_state(np.ascontiguousarray(U[:, :, ex.z0:ex.z1]))
        self.g.set_owned_rows(*ex.owned_local(), *ex.deep_local())

    def get_rows(self, buffer, k0, n, out):
        return self.g.get_rows(buffer, k0, n, out)

    def set_rows(self, buffer, k0, n, src):
        self.g.set_rows(buffer, k0, n, src)

    def push_rows(self, buffer, k0, n, dst, k0_dst):
        self.g.push_rows(buffer, k0, n, dst.g, k0_dst)

    def new_rows(self, n=GHOST):
        import torch
        return torch.empty((8, self.row_shape[1], n, self.row_shape[3]), dtype=torch.float64, device=self.device)

    def owned_state(self):
        """The rows of the global state this slab is responsible for (owned rows; plus the frozen boundary rows at
        the outer edges) and their global row offset."""
        ex = self.ext
        lo = 0 if ex.rank == 0 else ex.a
        hi = ex.nZ if ex.rank == ex.world - 1 else ex.b
        U = self.g.get_state()
        return lo, U[:, :, lo - ex.z0:hi - ex.z0]


def _make_buffer(slab, n):
    return slab.new_rows(n)


class SlabGroup:
    """All slabs of a run that live in THIS process: every rank (in-process driver) or this rank's one slab
    (torch.distributed driver, `dist` = the initialised torch.distributed module)."""

    def __init__(self, cfg, dt, U0, U, world, devices=("cuda:0",), dist=None, fused_exchange=True, **kw):
        self.cfg, self.world, self.dist = cfg, world, dist
        if dist is None:
            # linked slabs get a stream each: the stage kernels of different slabs are independent of each other (the
            # neighbours' streams are ordered between stages, clt_sync_peers), so on a shared GPU the last, partly filled
            # wave of one slab's kernel is topped up by the next slab's
            import torch
            streams = [torch.cuda.Stream(devices[r % len(devices)]) if fused_exchange and world > 1 else None for r in range(world)]
            self.slabs = [Slab(cfg, dt, U0, U, r, world, device=devices[r % len(devices)], stream=streams[r], **kw) for r in range(world)]
        else:
            self.slabs = [Slab(cfg, dt, U0, U, dist.get_rank(), world, device=devices[0], **kw)]
        self.extents = [s.ext for s in self.slabs]
        # slabs of one process: the stage kernels store the rows a neighbour needs straight into its ghost rows
        # (clt_link_rows: compute and exchange in one kernel); fused_exchange=False keeps the separate clt_push_rows kernels
        self.linked = dist is None and fused_exchange
        if self.linked:
            for lo, hi in zip(self.slabs[:-1], self.slabs[1:]):
                lo.g.link_rows(1, hi.g, *lo.ext.send_up(), hi.ext.recv_from_lower()[0])
                hi.g.link_rows(0, lo.g, *hi.ext.send_down(), lo.ext.recv_from_upper()[0])
                lo.g.sync_peers(hi.g)             # the neighbour's set-up is complete before anything is stored into its rows

    def step(self, n=1):
        for _ in range(n):
            for stage in (1, 2, 3, 4):
                for s in self.slabs:
                    s.g.step_stage(stage)
                if self.linked:
                    for lo, hi in zip(self.slabs[:-1], self.slabs[1:]):
                        lo.g.sync_peers(hi.g)          # stream order only (nothing to do on a shared stream)
                else:
                    exchange(self.slabs, self.extents, STAGE_BUFFER[stage], self.dist, _make_buffer)

    def step_cfl(self, n=1, cfl=0.0):
        """n adaptive RK4 steps (Fig. 3-4): every step runs with the global SETDT minimum of the state at
        its start.  Slabs of one process on one device keep dt on the device; across processes it is the minimum of the
        slabs' reductions (one MIN all-reduce and one host round trip per step).  Returns the time advanced."""
        if self.dist is None and n > 0 and len({str(s.device) for s in self.slabs}) == 1:
            # all slabs on one device: dt stays on the device (clt_cfl_open / clt_cfl_commit / clt_cfl_close) -- stage 4
            # collects each slab's minimum over its owned rows, one single-thread kernel takes the minimum over the slabs
            from . import clt
            ctxs = [s.g for s in self.slabs]
            for g in ctxs:
                g.cfl_open(cfl)
            clt.cfl_commit(ctxs, init=True)
            for _ in range(n):
                self.step(1)
                clt.cfl_commit(ctxs, init=False)
            return [g.cfl_close() for g in ctxs][0][1]
        t = 0.0
        for _ in range(n):
            dt = self.suggest_dt(cfl)
            for s in self.slabs:
                s.g.set_dt(dt)
            self.step(1)
            t += dt
        return t

    def diagnostics(self):
        """Global diagnostics: sums over the slabs' owned rows, max of the div B maxima."""
        parts = [s.g.diagnostics() for s in self.slabs]
        out = {k: sum(p[k] for p in parts) for k in ("kinetic", "magnetic", "magnetic_pert", "magnetic_n1")}
        out["max_divB"] = max(p["max_divB"] for p in parts)
        out["step"], out["time"] = parts[0]["step"], parts[0]["time"]
        if self.dist is not None:
            import torch
            dev = self.slabs[0].device
            t = torch.tensor([out[k] for k in ("kinetic", "magnetic", "magnetic_pert", "magnetic_n1")], dtype=torch.float64,
                             device=dev)
            m = torch.tensor([out["max_divB"]], dtype=torch.float64, device=dev)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM)
            self.dist.all_reduce(m, op=self.dist.ReduceOp.MAX)
            for k, v in zip(("kinetic", "magnetic", "magnetic_pert", "magnetic_n1"), t.tolist()):
                out[k] = v
            out["max_divB"] = float(m.item())
        return out

    def suggest_dt(self, cfl=0.0):
        dt = min(s.g.suggest_dt(cfl) for s in self.slabs)
        if self.dist is not None:
            import torch
            t = torch.tensor([dt], dtype=torch.float64, device=self.slabs[0].device)
            self.dist.all_reduce(t, op=self.dist.ReduceOp.MIN)
            dt = float(t.item())
        return dt

    def get_state(self):
        """The global state [8][nphi][nZ][nR] (in-process driver), or None on ranks > 0 (distributed: gathered on 0)."""
        pieces = [s.owned_state() for s in self.slabs]
        if self.dist is not None:
            gathered = [None] * self.world if self.dist.get_rank() == 0 else None
            self.dist.gather_object(pieces[0], gathered, dst=0)
            if self.dist.get_rank() != 0:
                return None
            pieces = gathered
        c = self.cfg
        U = np.empty((8, c.nphi, c.nZ, c.nR))
        for lo, block in pieces:
            U[:, :, lo:lo + block.shape[2]] = block
        return U

    def join(self):
        """Orders the first slab's stream after everything enqueued on the others' (for timing events on that stream)."""
        for s in self.slabs[1:]:
            self.slabs[0].g.sync_peers(s.g)

    def close(self):
        if self.linked:
            for s in self.slabs:                  # no dangling peer pointers while contexts go away one by one
                s.g.link_rows(0, None)
                s.g.link_rows(1, None)
        for s in self.slabs:
            s.g.close()
