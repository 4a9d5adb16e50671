"""x-slab sharding of the SSP-RK3 step across ranks.

The phase-space grid is cut into contiguous slabs of x-elements, one per rank; the velocity axes stay
whole, so the density moment (Eq. 27) is local.  Per Runge-Kutta stage:

  1. rho of the own x nodes                       (dg_density, local -- or, from the second stage of a run on, the
     density the previous stage's dg_rk_stage finished from its kernel-epilogue partials: no extra pass over f)
  2. all-gather of rho (N_x n_x doubles, 4 KB at 512^3); every rank then solves the same global
     Fourier-series Poisson problem (Eq. 63 / 71) and keeps E at its own nodes --
     bit-identical to the unsharded solve, whatever the number of ranks
  3. face-plane exchange with the two x-neighbours: the upwind flux (Eq. 23) at a slab's
     first / last x face needs the neighbour's last / first x-node plane (N_u n_u x N_v n_v doubles,
     2.1 MB at 512^3), sent straight out of the stage array, received into the halo buffer the kernels
     read (dg_set_xhalo)
  4. fused RHS + stage combination              (dg_rk_stage, local)

With `push=True` step 3 disappears as a separate operation: every rank's dg_rk_stage stores the two boundary planes of
its OUTPUT straight into the neighbours' halo buffers from inside the RHS kernel (dg_set_xhalo_push: peer memory over
NVLink, symmetric-memory allocation), into the buffer of the other parity than the one the running stage reads; the
all-gather of step 2 is then the only thing that orders the ranks between two stages.

This module is host plumbing only: which planes go where, and in what order the C-ABI calls and the
torch.distributed calls are issued (the stage coefficients too come from the backend: dg_ssprk3_stage_coeffs).  The arithmetic runs behind the `backend` object -- `CudaBackend`
(libdgvlasov kernels) in the product; there is no CPU backend here, and constructing `CudaBackend`
without a CUDA device raises.  The CPU tests drive the same plumbing over gloo with a backend of their
own (tests/_xslab_worker.py).
"""
from __future__ import annotations

import torch
import torch.distributed as dist

def slab_partition(n_elem_x: int, world: int):
    """[(e0, e1)] per rank: contiguous, sizes differ by at most one element, every rank non-empty."""
    if world < 1 or n_elem_x < world:
        raise ValueError(f"cannot cut {n_elem_x} x-elements into {world} non-empty slabs")
    return [(r * n_elem_x // world, (r + 1) * n_elem_x // world) for r in range(world)]


def slab_bounds(lo_x: float, hi_x: float, n_elem_x: int, e0: int, e1: int):
    dx = (hi_x - lo_x) / n_elem_x
    return lo_x + e0 * dx, lo_x + e1 * dx


class TorchDistComm:
    """The two collectives of the sharded step over torch.distributed (NCCL on GPUs, gloo in the CPU tests).
    With world == 1 (no process group) both degenerate to local copies."""

    def __init__(self, rank: int, world: int, group=None):
        self.rank, self.world, self.group = rank, world, group
        if world > 1 and not dist.is_initialized():
            raise RuntimeError("TorchDistComm: world > 1 needs an initialised process group")

    def exchange_faces(self, first_plane, last_plane, halo, periodic: bool):
        """halo[0] <- left neighbour's last plane, halo[1] <- right neighbour's first plane.
        Non-periodic x: the outermost ranks get zeros (zero inflow, reading C2)."""
        r, w = self.rank, self.world
        if w == 1:
            if periodic:
                halo[0].copy_(last_plane); halo[1].copy_(first_plane)
            else:
                halo.zero_()
            return
        left, right = (r - 1) % w, (r + 1) % w
        has_left, has_right = periodic or r > 0, periodic or r < w - 1
        ops = []
        # tag 0: "a last plane travelling right", tag 1: "a first plane travelling left".  Sends and receives are
        # posted in the same order on every rank, so two ranks that are each other's left AND right neighbour match up.
        if has_right:
            ops.append(dist.P2POp(dist.isend, last_plane, right, self.group, 0))
        if has_left:
            ops.append(dist.P2POp(dist.isend, first_plane, left, self.group, 1))
        if has_left:
            ops.append(dist.P2POp(dist.irecv, halo[0], left, self.group, 0))
        else:
            halo[0].zero_()
        if has_right:
            ops.append(dist.P2POp(dist.irecv, halo[1], right, self.group, 1))
        else:
            halo[1].zero_()
        for work in dist.batch_isend_irecv(ops):
            work.wait()

    def alloc_halos(self, plane_shape, device, periodic: bool):
        """Ping-pong halo buffers [parity][side][G_u][G_v] for the fused face push, plus views of the two x-neighbours'
        buffers (None where there is no neighbour).  world == 1: the neighbour is this rank itself.  world > 1: the
        buffers live in symmetric memory so that every rank can store into its neighbours' over NVLink."""
        shape = (2, 2) + tuple(plane_shape)
        r, w = self.rank, self.world
        if w == 1:
            own = torch.zeros(shape, dtype=torch.float64, device=device)
            return own, (own if periodic else None), (own if periodic else None)
        try:
            import torch.distributed._symmetric_memory as symm
        except Exception as e:                                      # pragma: no cover
            raise RuntimeError("push mode with world > 1 needs torch.distributed._symmetric_memory") from e
        own = symm.empty(shape, dtype=torch.float64, device=device)
        own.zero_()
        hdl = symm.rendezvous(own, self.group if self.group is not None else dist.group.WORLD)
        left = hdl.get_buffer((r - 1) % w, shape, torch.float64) if (periodic or r > 0) else None
        right = hdl.get_buffer((r + 1) % w, shape, torch.float64) if (periodic or r < w - 1) else None
        return own, left, right

    def device_barrier(self, token):
        """Orders the ranks' streams when no all-gather does (runs without a field solve)."""
        if self.world > 1:
            dist.all_reduce(token, group=self.group)

    def all_gather_rho(self, rho_loc, counts, out):
        """out[G_x] <- concatenation of every rank's rho (counts[r] nodes each; padded to the longest slab on the wire)."""
        if self.world == 1:
            out.copy_(rho_loc)
            return out
        m = max(counts)
        send = rho_loc if rho_loc.numel() == m else torch.cat([rho_loc, rho_loc.new_zeros(m - rho_loc.numel())])
        buf = rho_loc.new_empty(self.world * m)
        dist.all_gather_into_tensor(buf, send.contiguous(), group=self.group)
        off = 0
        for r, c in enumerate(counts):
            out[off:off + c].copy_(buf[r * m:r * m + c])
            off += c
        return out


class HostStagedComm(TorchDistComm):
    """The same two collectives with every message staged through host memory, over a CPU process group (gloo).
    For ranks that cannot talk NCCL to each other -- above all several ranks sharing ONE GPU (NCCL refuses duplicate
    devices), which is how the sharded step is exercised as concurrent processes on a single-GPU box.  Each transfer
    synchronises the rank's stream (the .cpu() copies), so no kernel ever waits for another process's kernel; the ranks
    meet in gloo on the host.  Plain exchange only: the fused face push needs peer-mapped halo buffers."""

    def exchange_faces(self, first_plane, last_plane, halo, periodic: bool):
        if self.world == 1:
            return super().exchange_faces(first_plane, last_plane, halo, periodic)
        r, w = self.rank, self.world
        left, right = (r - 1) % w, (r + 1) % w
        has_left, has_right = periodic or r > 0, periodic or r < w - 1
        first_h, last_h = first_plane.cpu().contiguous(), last_plane.cpu().contiguous()
        in_l, in_r = torch.empty_like(first_h), torch.empty_like(first_h)
        ops = []
        if has_right:
            ops.append(dist.P2POp(dist.isend, last_h, right, self.group, 0))
        if has_left:
            ops.append(dist.P2POp(dist.isend, first_h, left, self.group, 1))
        if has_left:
            ops.append(dist.P2POp(dist.irecv, in_l, left, self.group, 0))
        if has_right:
            ops.append(dist.P2POp(dist.irecv, in_r, right, self.group, 1))
        for work in dist.batch_isend_irecv(ops):
            work.wait()
        halo[0].copy_(in_l) if has_left else halo[0].zero_()
        halo[1].copy_(in_r) if has_right else halo[1].zero_()

    def alloc_halos(self, plane_shape, device, periodic: bool):
        if self.world == 1:
            return super().alloc_halos(plane_shape, device, periodic)
        raise RuntimeError("HostStagedComm: the fused face push needs peer-mapped halo buffers (use TorchDistComm over NCCL)")

    def device_barrier(self, token):
        if self.world > 1:
            torch.cuda.synchronize(token.device) if token.is_cuda else None
            dist.barrier(group=self.group)

    def all_gather_rho(self, rho_loc, counts, out):
        if self.world == 1:
            return super().all_gather_rho(rho_loc, counts, out)
        m = max(counts)
        send = torch.zeros(m, dtype=rho_loc.dtype)
        send[:rho_loc.numel()].copy_(rho_loc)                       # device -> host (synchronises the stream)
        buf = torch.empty(self.world * m, dtype=rho_loc.dtype)
        dist.all_gather_into_tensor(buf, send, group=self.group)
        off = 0
        for r, c in enumerate(counts):
            out[off:off + c].copy_(buf[r * m:r * m + c])
            off += c
        return out


class CudaBackend:
    """The arithmetic of one slab, through the C ABI: a slab context (bc[0] = DG_BC_HALO) for density and the fused
    RHS + stage kernel, and an x-only context over the GLOBAL grid for the Poisson solve."""

    def __init__(self, nelem, order, lo, hi, bc, omega_c, pmax, mass_mode, e0, e1, device):
        if not torch.cuda.is_available():
            raise RuntimeError("CudaBackend: no CUDA device (the DG kernels have no CPU fallback)")
        from . import api
        self.api = api
        self.device = torch.device("cuda", device)
        lo_s, hi_s = slab_bounds(lo[0], hi[0], nelem[0], e0, e1)
        nel = (e1 - e0,) + tuple(nelem[1:])
        self.slab = api.DGContext(nel, order, (lo_s,) + tuple(lo[1:]), (hi_s,) + tuple(hi[1:]),
                                  bc=(api.BC_HALO,) + tuple(bc[1:]), omega_c=omega_c, pmax=1, mass_mode=mass_mode, device=device)
        self.field = api.DGContext((nelem[0],), (order[0],), (lo[0],), (hi[0],), pmax=pmax, mass_mode=mass_mode, device=device)
        self.flat_shape = self.slab.flat_shape

    def empty(self, shape):
        return torch.empty(shape, dtype=torch.float64, device=self.device)

    def density(self, f, out):
        return self.slab.density(f, out)

    def poisson_E(self, rho, out):
        return self.field.poisson_E(rho, out)

    def set_halo(self, halo):
        self.slab.set_xhalo(halo)

    def rk_stage(self, f_s, f_n, E_loc, out, c0, c1, dt, rho_out=None):
        return self.slab.rk_stage(f_s, f_n, E_loc, out, c0, c1, dt, rho_out)

    def set_push(self, left_dst, right_dst):
        self.slab.set_xhalo_push(left_dst, right_dst)

    def plain_launches(self):
        """Push mode across devices: no programmatic dependent launch around the collectives that order the peer stores
        (point 3)."""
        self.slab.set_option(self.api.OPT_PDL, 0)
        self.field.set_option(self.api.OPT_PDL, 0)

    def stage_coeffs(self, stage):
        """(c0, c1) of Shu-Osher stage 0, 1, 2: the table lives in the library (dg_ssprk3_stage_coeffs)."""
        return self.api.ssprk3_stage_coeffs(stage)

    def close(self):
        self.slab.close(); self.field.close()


class XSlabStepper:
    """SSP-RK3 on one x-slab.  `f` is this rank's slab [G_x_local][G_u][G_v] (device tensor for CudaBackend)."""

    def __init__(self, nelem, order, lo, hi, bc=None, omega_c=0.0, pmax=0, mass_mode=0, rank=0, world=1, device=0,
                 backend=None, comm=None, push=False):
        ndim = len(nelem)
        self.bc = tuple(bc) if bc is not None else (0,) + (1,) * (ndim - 1)
        self.parts = slab_partition(nelem[0], world)
        self.e0, self.e1 = self.parts[rank]
        self.n0 = order[0]
        self.counts = [(b - a) * self.n0 for a, b in self.parts]
        self.g0, self.g1 = self.e0 * self.n0, self.e1 * self.n0
        self.G0 = nelem[0] * self.n0
        self.rank, self.world = rank, world
        self.be = backend if backend is not None else CudaBackend(nelem, order, lo, hi, self.bc, omega_c, pmax, mass_mode,
                                                                  self.e0, self.e1, device)
        self.comm = comm if comm is not None else TorchDistComm(rank, world)
        shp = tuple(self.be.flat_shape)
        self.u1, self.u2 = self.be.empty(shp), self.be.empty(shp)
        self.push = bool(push)
        if self.push:
            # [parity][side][G_u][G_v]; stage number `sidx` reads parity sidx % 2 and pushes into the neighbours' other one
            self.H, self.H_left, self.H_right = self.comm.alloc_halos(shp[1:], self.u1.device, periodic=(self.bc[0] == 0))
            self.sidx = 0
            self.halo = self.H[0]
            if world > 1 and hasattr(self.be, "plain_launches"):
                self.be.plain_launches()
            self.token = self.be.empty((1,))
        else:
            self.halo = self.be.empty((2,) + shp[1:])
        self.be.set_halo(self.halo)
        self.rho_loc, self.rho = self.be.empty((shp[0],)), self.be.empty((self.G0,))
        self.E = self.be.empty((self.G0,))
        self.E_loc = self.be.empty((shp[0],))

    def field(self, f_s, rho_known=False):
        """Steps 1-2: E at the own x nodes from the global density.  rho_known: self.rho_loc already holds the density
        of f_s (written by the previous stage's rk_stage)."""
        if not rho_known:
            self.be.density(f_s, self.rho_loc)
        self.comm.all_gather_rho(self.rho_loc, self.counts, self.rho)
        self.be.poisson_E(self.rho, self.E)
        self.E_loc.copy_(self.E[self.g0:self.g1])
        return self.E_loc

    def stage(self, f_s, f_n, out, c0, c1, dt, self_consistent=True, rho_known=False):
        """One stage; with self_consistent the density of `out` is left in self.rho_loc for the next stage.
        rho_known also says that the previous stage of this stepper produced f_s (push mode: its faces are in the halos)."""
        E = self.field(f_s, rho_known) if self_consistent else None
        if self.push:
            cur, nxt = self.sidx % 2, (self.sidx + 1) % 2
            self.halo = self.H[cur]
            if not rho_known:          # f_s did not come from the previous stage: fill this parity by a plain exchange
                self.comm.exchange_faces(f_s[0], f_s[-1], self.halo, periodic=(self.bc[0] == 0))
            elif not self_consistent:  # no all-gather between the stages: order the ranks explicitly
                self.comm.device_barrier(self.token)
            self.be.set_halo(self.halo)
            self.be.set_push(None if self.H_left is None else self.H_left[nxt][1],
                             None if self.H_right is None else self.H_right[nxt][0])
            self.sidx += 1
        else:
            self.comm.exchange_faces(f_s[0], f_s[-1], self.halo, periodic=(self.bc[0] == 0))
        self.be.rk_stage(f_s, f_n if c0 != 0.0 else None, E, out, c0, c1, dt, self.rho_loc if self_consistent else None)
        return out

    def step(self, f, dt, self_consistent=True, rho_known=False):
        """u1 = u + dt L(u); u2 = 3/4 u + 1/4 (u1 + dt L(u1)); u <- 1/3 u + 2/3 (u2 + dt L(u2)), in place.
        rho_known is for run(): a lone step cannot know whether the caller touched f since the last one."""
        (a0, b0), (a1, b1), (a2, b2) = (self.be.stage_coeffs(s) for s in range(3))     # method arithmetic stays behind the backend
        self.stage(f, f, self.u1, a0, b0, dt, self_consistent, rho_known)
        self.stage(self.u1, f, self.u2, a1, b1, dt, self_consistent, True)
        self.stage(self.u2, f, f, a2, b2, dt, self_consistent, True)
        return f

    def run(self, f, dt, nsteps, self_consistent=True):
        for i in range(nsteps):
            self.step(f, dt, self_consistent, rho_known=(i > 0))
        return f

    def close(self):
        if hasattr(self.be, "close"):
            self.be.close()
