"""Uniform-grid stepper on top of the C-ABI calls: the "whole hot path" that bench.py times.

One step (collapsed onto the GPU):
    srhd_max_signal_speed(grid)          K2 of the paper: the CFL reduction (Eq. 26-28)
    dt = C_CFL * dh / S_max              one double crosses to the host (Eq. 28, formed by the caller)
    srhd_grid_gather(grid) -> tiles      ghost-zone fill of every 16^3 patch group (stands in for P:219)
    srhd_fluid_step(tiles) -> patches    K1 of the paper: the fused MUSCL-Hancock update
    srhd_grid_scatter(patches) -> grid

Nothing here computes on the host except the scalar division for dt; all buffers are torch CUDA
tensors allocated once.  There is no CPU fallback.
"""
import numpy as np
import torch

from . import binding as B


class GridStepper:
    """Owns the device buffers of one uniform grid (5, nz, ny, nx) of conserved variables."""

    def __init__(self, shape, dh, bc, recon="plm", riemann="hllc", cfl=0.4, inflow=None, exact=False,
                 device="cuda", dt_speed="signal", **par_overrides):
        nz, ny, nx = shape
        if nx % 16 or ny % 16 or nz % 16:
            raise B.SrhdError("grid extents must be multiples of 16 (whole patch groups)")
        self.shape, self.dh, self.bc, self.cfl, self.exact = (nz, ny, nx), float(dh), list(bc), float(cfl), exact
        self.par = B.params(recon, riemann, exact=exact, **par_overrides)
        if dt_speed not in ("signal", "light"):
            raise B.SrhdError("dt_speed must be 'signal' (Eq. 26-28) or 'light' (S_max replaced by c, P:229)")
        self.dt_speed = dt_speed
        self.npg = (nx // 16) * (ny // 16) * (nz // 16)
        self.ncell = nx * ny * nz
        nxt = 16 + 2 * self.par.ghost
        f64 = dict(dtype=torch.float64, device=device)
        self.grid = torch.empty((5, nz, ny, nx), **f64)
        self.tiles = torch.empty((self.npg, 5, nxt, nxt, nxt), **f64)
        self.patches = torch.empty((self.npg, 8, 5, 8, 8, 8), **f64)
        self.smax = torch.zeros(1, **f64)
        self.stats = B.new_stats(device)
        self.inflow = None
        if inflow is not None:      # (mask (ny,nx) uint8, conserved inflow state, 5 floats)
            mask, cons = inflow
            self.inflow = (torch.as_tensor(np.ascontiguousarray(mask, dtype=np.uint8)).to(device),
                           [float(v) for v in cons])
        # the fixed-inflow ghost cells take part in the update, so their signal speed bounds dt too
        # (Eq. 28 over every state of the stencil); one srhd_max_signal_speed call on that one state
        self.smax_inflow = 0.0
        if self.inflow is not None:
            c = torch.tensor(self.inflow[1], **f64).reshape(5, 1).contiguous()
            self.smax_inflow = float(B.max_signal_speed(c, self.par, exact=exact).cpu())
        self.t = 0.0
        self.nstep = 0
        self._smax_fresh = False   # True when self.smax holds S_max of self.grid (written by the fused scatter)
        self.launches_per_step = 4 if dt_speed == "signal" else 3   # gather, fluid step, scatter(+speed), smax finish

    # ---- state in / out -------------------------------------------------------------------------
    def set_prim(self, prim):
        """Upload a primitive field (5,nz,ny,nx) (numpy or CUDA tensor) and convert with srhd_prim2cons."""
        p = prim if isinstance(prim, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(prim))
        p = p.to(self.grid.device).reshape(5, -1).contiguous()
        B.prim2cons(p, cons=self.grid.view(5, -1), exact=self.exact)
        self._smax_fresh = False
        return self

    def set_cons(self, cons):
        c = cons if isinstance(cons, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(cons))
        self.grid.copy_(c.reshape(self.grid.shape), non_blocking=True)
        self._smax_fresh = False
        return self

    def prim(self):
        """Primitive field of the current state via srhd_cons2prim (device tensor (5,nz,ny,nx))."""
        w, _ = B.cons2prim(self.grid.view(5, -1), self.par, exact=self.exact)
        return w.view(self.grid.shape)

    # ---- one step -------------------------------------------------------------------------------
    def signal_speed(self):
        if self.dt_speed == "light":           # the conservative CFL condition, no reduction kernel
            return 1.0
        if self._smax_fresh:                   # the previous step's scatter already reduced this state
            return max(float(self.smax.cpu()), self.smax_inflow)
        B.max_signal_speed(self.grid.view(5, -1), self.par, out=self.smax, exact=self.exact)
        return max(float(self.smax.cpu()), self.smax_inflow)   # the one device->host double per step

    def advance(self, dt, kernel_events=None):
        """gather -> fluid_step -> scatter with a given dt (asynchronous on the current stream).
        kernel_events: a list that receives a (start, end) CUDA event pair around srhd_fluid_step."""
        B.grid_gather(self.grid, self.par.ghost, self.bc, self.inflow, cons_in=self.tiles, exact=self.exact)
        if kernel_events is not None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
        B.fluid_step(self.tiles, dt, self.dh, self.par, cons_out=self.patches, stats=self.stats,
                     exact=self.exact)
        if kernel_events is not None:
            e1.record()
            kernel_events.append((e0, e1))
        if self.dt_speed == "signal":          # scatter fused with the CFL reduction of the new state
            B.grid_scatter_speed(self.patches, self.shape, self.par, grid=self.grid, out=self.smax, exact=self.exact)
            self._smax_fresh = True
        else:
            B.grid_scatter(self.patches, self.shape, grid=self.grid, exact=self.exact)
        self.t += dt
        self.nstep += 1

    def step(self, t_end=None, kernel_events=None):
        """One full step: CFL reduction, dt (clipped to hit t_end exactly), update.  Returns dt."""
        dt = self.cfl * self.dh / self.signal_speed()
        if t_end is not None and self.t + dt > t_end:
            dt = t_end - self.t
        self.advance(dt, kernel_events)
        return dt

    def step_async(self, kernel_events=None):
        """One full step with NO host synchronisation: dt = C dh / S_max is formed on the device by
        srhd_fluid_step_cfl from the speed the previous scatter (or a CFL kernel) left there.  The
        host does not learn dt, so self.t is not advanced: use step() when the time matters."""
        if self.dt_speed == "light":
            return self.advance(self.cfl * self.dh, kernel_events)
        if not self._smax_fresh:
            B.max_signal_speed(self.grid.view(5, -1), self.par, out=self.smax, exact=self.exact)
        B.grid_gather(self.grid, self.par.ghost, self.bc, self.inflow, cons_in=self.tiles, exact=self.exact)
        if kernel_events is not None:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
        B.fluid_step_cfl(self.tiles, self.cfl, self.dh, self.smax, self.par, min_speed=self.smax_inflow,
                         cons_out=self.patches, stats=self.stats, exact=self.exact)
        if kernel_events is not None:
            e1.record()
            kernel_events.append((e0, e1))
        # the fluid step has read self.smax (stream order), the fused scatter may now overwrite it
        B.grid_scatter_speed(self.patches, self.shape, self.par, grid=self.grid, out=self.smax, exact=self.exact)
        self._smax_fresh = True
        self.nstep += 1

    def run(self, nsteps=None, t_end=None):
        n = 0
        while (nsteps is None or n < nsteps) and (t_end is None or self.t < t_end):
            self.step(t_end)
            n += 1
        return n

    def last_stats(self):
        return B.stats_to_host(self.stats)
