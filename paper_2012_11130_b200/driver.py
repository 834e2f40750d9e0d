"""Uniform-grid stepper on top of the C-ABI calls: the "whole hot path" that bench.py times.

The state lives in the PATCH layout the solver writes (cons_out of srhd_fluid_step: 8^3 patches, as in
the paper's AMR code); a uniform grid (5, nz, ny, nx) is only materialised when it is asked for.
One step (collapsed onto the GPU):
    srhd_patch_gather_speed(patches) -> tiles, S_max   ghost-zone fill of every 16^3 patch group from the
                                                       neighbouring patches (stands in for P:219) fused
                                                       with the CFL reduction of that state (Eq. 26-27)
    srhd_fluid_step_cfl(tiles) -> patches              the fused MUSCL-Hancock update with
                                                       dt = C dh / S_max formed on the device (Eq. 28)
step_async() issues both behind ONE call, srhd_grid_step_cfl (4 launches, patches double buffered), whose first
kernel also finishes the patch groups that hold a single state (their new patches are their old ones) without
ever materialising their tiles; fused=False keeps the two separate calls (same results bit for bit).
The first step after set_prim / set_cons starts from the grid instead: srhd_max_signal_speed +
srhd_grid_gather.  step() reads S_max back (one double) because the host wants t; step_async() does not
synchronise.  Nothing here computes on the host except that scalar arithmetic; all buffers are torch
CUDA tensors allocated once.  There is no CPU fallback.
"""
import numpy as np
import torch

from . import binding as B


class GridStepper:
    """Owns the device buffers of one uniform grid of conserved variables."""

    def __init__(self, shape, dh, bc, recon="plm", riemann="hllc", cfl=0.4, inflow=None, exact=False,
                 device="cuda", dt_speed="signal", fused=True, **par_overrides):
        nz, ny, nx = shape
        if nx % 16 or ny % 16 or nz % 16:
            raise B.SrhdError("grid extents must be multiples of 16 (whole patch groups)")
        self.shape, self.dh, self.bc, self.cfl, self.exact = (nz, ny, nx), float(dh), list(bc), float(cfl), exact
        self.par = B.params(recon, riemann, exact=exact, **par_overrides)
        if dt_speed not in ("signal", "light"):
            raise B.SrhdError("dt_speed must be 'signal' (Eq. 26-28) or 'light' (S_max replaced by c, P:229)")
        self.dt_speed = dt_speed
        self.fused = bool(fused)   # step_async() through srhd_grid_step_cfl (False: the two separate calls)
        self.npg = (nx // 16) * (ny // 16) * (nz // 16)
        self.ncell = nx * ny * nz
        nxt = 16 + 2 * self.par.ghost
        B.load_library(exact)
        f64 = dict(dtype=B._CUR_REAL, device=device)   # srhd_real of the selected library (float32 for the f32 builds)
        self._grid = torch.empty((5, nz, ny, nx), **f64)
        self.tiles = torch.empty((self.npg, 5, nxt, nxt, nxt), **f64)
        self.patches = torch.empty((self.npg, 8, 5, 8, 8, 8), **f64)
        self._patches_b = None    # second patch buffer, allocated by the first fused step (srhd_grid_step_cfl)
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
        self._in_patches = False   # True: self.patches holds the current state (self._grid may be stale)
        self._grid_stale = False
        # fused: own-uniform flags, pre-pass (ghost-zone fill + speed + uniform tiles), smax finish, march; else
        # gather + speed, smax finish, uniform-tile scan, march
        self.launches_per_step = 4

    # ---- state in / out -------------------------------------------------------------------------
    @property
    def grid(self):
        """The current state as a uniform grid (5,nz,ny,nx); scattered from the patches on demand."""
        if self._grid_stale:
            B.grid_scatter(self.patches, self.shape, grid=self._grid, exact=self.exact)
            self._grid_stale = False
        return self._grid

    def set_prim(self, prim):
        """Upload a primitive field (5,nz,ny,nx) (numpy or CUDA tensor) and convert with srhd_prim2cons."""
        p = prim if isinstance(prim, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(prim))
        p = p.to(self._grid.device, dtype=self._grid.dtype).reshape(5, -1).contiguous()
        B.prim2cons(p, cons=self._grid.view(5, -1), exact=self.exact)
        self._in_patches = self._grid_stale = False
        return self

    def set_cons(self, cons):
        c = cons if isinstance(cons, torch.Tensor) else torch.from_numpy(np.ascontiguousarray(cons))
        self._grid.copy_(c.reshape(self._grid.shape), non_blocking=True)
        self._in_patches = self._grid_stale = False
        return self

    def prim(self):
        """Primitive field of the current state via srhd_cons2prim (device tensor (5,nz,ny,nx))."""
        w, _ = B.cons2prim(self.grid.view(5, -1), self.par, exact=self.exact)
        return w.view(self._grid.shape)

    # ---- one step -------------------------------------------------------------------------------
    def _fill_tiles(self, need_speed):
        """Ghost-zone fill of the current state into self.tiles; S_max of it into self.smax if asked."""
        if self._in_patches:
            # fused: tiles from the neighbouring patches + CFL reduction (the speed costs nothing extra to skip)
            B.patch_gather_speed(self.patches, self.shape, self.par, self.bc, self.inflow, cons_in=self.tiles,
                                 out=self.smax, exact=self.exact)
        else:
            if need_speed:
                B.max_signal_speed(self._grid.view(5, -1), self.par, out=self.smax, exact=self.exact)
            B.grid_gather(self._grid, self.par.ghost, self.bc, self.inflow, cons_in=self.tiles, exact=self.exact)

    def _timed(self, kernel_events, launch):
        if kernel_events is None:
            return launch()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        launch()
        e1.record()
        kernel_events.append((e0, e1))

    def _done(self):
        self._in_patches = self._grid_stale = True
        self.nstep += 1

    def advance(self, dt, kernel_events=None):
        """Ghost-zone fill -> srhd_fluid_step with a given dt (asynchronous on the current stream)."""
        self._fill_tiles(need_speed=False)
        self._timed(kernel_events, lambda: B.fluid_step(self.tiles, dt, self.dh, self.par, cons_out=self.patches,
                                                        stats=self.stats, exact=self.exact))
        self.t += dt
        self._done()

    def step(self, t_end=None, kernel_events=None):
        """One full step with dt on the host: CFL reduction, dt (clipped to hit t_end exactly), update."""
        if self.dt_speed == "light":           # the conservative CFL condition, no reduction
            smax = 1.0
        else:
            self._fill_tiles(need_speed=True)
            smax = max(float(self.smax.cpu()), self.smax_inflow)   # the one device->host double per step
            if not (0.0 < smax <= 1.0):   # a NaN / vacuum state somewhere: the max-reduction cannot speak for it
                raise B.SrhdError(f"signal speed {smax!r} is not in (0, 1]: the state holds non-finite or unphysical cells "
                                  f"(srhd_stats of the last step: {self.last_stats().algorithm_dict()})")
        dt = self.cfl * self.dh / smax
        if t_end is not None and self.t + dt > t_end:
            dt = t_end - self.t
        if self.dt_speed == "light":
            self.advance(dt, kernel_events)
            return dt
        self._timed(kernel_events, lambda: B.fluid_step(self.tiles, dt, self.dh, self.par, cons_out=self.patches,
                                                        stats=self.stats, exact=self.exact))
        self.t += dt
        self._done()
        return dt

    def step_async(self, kernel_events=None):
        """One full step with NO host synchronisation: dt = C dh / S_max is formed on the device by
        srhd_fluid_step_cfl.  The host does not learn dt, so self.t is not advanced: use step() when
        the time matters."""
        if self.dt_speed == "light":
            return self.advance(self.cfl * self.dh, kernel_events)
        if self._in_patches and self.fused:
            # the whole step behind one call: uniform patch groups are finished by its first kernel straight
            # from the patches (no tile), the others are gathered and marched; patches are double buffered
            if self._patches_b is None:
                self._patches_b = torch.empty_like(self.patches)
            self._timed(kernel_events, lambda: B.grid_step_cfl(
                self.patches, self._patches_b, self.tiles, self.shape, self.cfl, self.dh, self.par, self.bc,
                self.inflow, min_speed=self.smax_inflow, stats=self.stats, out=self.smax, exact=self.exact))
            self.patches, self._patches_b = self._patches_b, self.patches
            return self._done()
        self._fill_tiles(need_speed=True)
        self._timed(kernel_events, lambda: B.fluid_step_cfl(self.tiles, self.cfl, self.dh, self.smax, self.par,
                                                            min_speed=self.smax_inflow, cons_out=self.patches,
                                                            stats=self.stats, exact=self.exact))
        self._done()

    def signal_speed(self):
        """S_max of the current state (Eq. 26-27, bounded below by the inflow state's) on the host."""
        if self.dt_speed == "light":
            return 1.0
        B.max_signal_speed(self.grid.view(5, -1), self.par, out=self.smax, exact=self.exact)
        return max(float(self.smax.cpu()), self.smax_inflow)

    def run(self, nsteps=None, t_end=None):
        n = 0
        while (nsteps is None or n < nsteps) and (t_end is None or self.t < t_end):
            self.step(t_end)
            n += 1
        return n

    def last_stats(self):
        return B.stats_to_host(self.stats)
