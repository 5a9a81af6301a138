"""Time stepping of the fluid solver on a box, as sequences of libfsei calls (plumbing only: no arithmetic here).

One time step of the paper's scheme (Eq. 3; V1) is one substep (Adams-Bashforth, gamma = 3/2,
rho = -1/2) or three (the low-storage third-order Runge-Kutta scheme of the paper's refs [12],[13]:
gamma = (8/15, 5/12, 3/4), rho = (0, -17/60, -5/12), alpha_l = gamma_l + rho_l); a substep is

    without markers:  fsei_fluid_substep  (explicit terms -> implicit viscous step -> pressure projection)
    with markers:     fsei_ibm_forcing -> fsei_explicit_terms (no body force) -> fsei_ibm_apply_forcing (rhs += alpha dt f on the
                      markers' supports, which also clears f) -> fsei_viscous_step -> fsei_pressure_projection
                      -- the forcing fields are zero-filled once and never streamed as a whole again

with beta_l = alpha_l dt / (2 Re).  The first Adams-Bashforth step has no H^{n-1} and runs as forward Euler
(gamma = 1, rho = 0).  All fields live on the device; nothing synchronises, so a step can be captured in a CUDA graph.
"""
from __future__ import annotations

SCHEMES = {
    "ab2": ((1.5,), (-0.5,)),
    "rk3": ((8.0 / 15.0, 5.0 / 12.0, 3.0 / 4.0), (0.0, -17.0 / 60.0, -5.0 / 12.0)),
}


class FluidStepper:
    def __init__(self, plan, u, v, w, dt: float, Re: float, scheme: str = "rk3", markers=None):
        """plan: binding.Plan; u, v, w: device float64 tensors [nz][ny][nx] (updated in place).
        markers: optional dict of device tensors xm, ym, zm, area, Vu, Vv, Vw (an immersed body moving with velocity V)."""
        import torch
        if scheme not in SCHEMES:
            raise ValueError(f"scheme must be one of {sorted(SCHEMES)}")
        self.plan, self.dt, self.Re, self.scheme = plan, float(dt), float(Re), scheme
        self.u, self.v, self.w = u, v, w
        z = lambda: torch.zeros_like(u)
        self.p, self.phi = z(), z()
        self.h = [z(), z(), z()]                       # H of the previous substep
        self.r = [z(), z(), z()]                       # scratch: right-hand sides
        self.markers = markers
        if markers is not None:
            n = markers["xm"].shape[0]
            self.f = [z(), z(), z()]
            self.F = [torch.zeros(n, dtype=u.dtype, device=u.device) for _ in range(3)]
        self.steps = 0
        self.launches = 0
        self._graph = None

    def substep(self, gamma: float, rho: float, stream=None):
        dt, alpha = self.dt, gamma + rho
        beta = alpha * dt / (2.0 * self.Re)
        P = self.plan
        if self.markers is None:
            P.fluid_substep(self.u, self.v, self.w, self.p, *self.h, *self.r, self.phi, gamma * dt, rho * dt, alpha * dt, beta,
                            stream=stream)
            self.launches += P.last_launch_count
            return
        m = self.markers
        n = m["xm"].shape[0]
        P.ibm_forcing(n, m["xm"], m["ym"], m["zm"], m["area"], m["Vu"], m["Vv"], m["Vw"], self.u, self.v, self.w,
                      1.0 / (alpha * dt), *self.F, *self.f, stream=stream)
        self.launches += P.last_launch_count
        P.explicit_terms(self.u, self.v, self.w, self.p, *self.h, *self.r, gamma * dt, rho * dt, alpha * dt, beta, stream=stream)
        self.launches += P.last_launch_count
        P.ibm_apply_forcing(n, m["xm"], m["ym"], m["zm"], *self.f, *self.r, alpha * dt, stream=stream)
        self.launches += P.last_launch_count
        P.viscous_step(self.u, self.v, self.w, *self.r, beta, stream=stream)
        self.launches += P.last_launch_count
        P.pressure_projection(self.u, self.v, self.w, self.p, self.phi, alpha * dt, beta, stream=stream)
        self.launches += P.last_launch_count

    def step(self, stream=None):
        gam, rho = SCHEMES[self.scheme]
        if self.scheme == "ab2" and self.steps == 0:
            gam, rho = (1.0,), (0.0,)                  # no H^{n-1} yet: forward Euler
        for g, r in zip(gam, rho):
            self.substep(g, r, stream)
        self.steps += 1

    def capture(self):
        """Capture one whole time step (all its substeps: every launch of every call) in a CUDA graph; `replay()` then runs a
        step with one graph launch instead of 10-30 kernel launches per substep.  Measured on B200 (RK3 step): 32^3 0.50 -> 0.46 ms
        (54 launches: the kernels themselves are latency-bound there), 256^3 no difference -- the eager path was not waiting on the
        host; the graph is for callers that want ONE launch per step (serving loops, overlap with other streams).  Call after at least one eager step.  The graph holds the
        field pointers and dt, Re, the scheme and the markers' arrays as they are now (marker POSITIONS may be updated in place
        between replays).  The capture itself advances the solution by one step."""
        import torch
        if self.steps == 0:
            raise RuntimeError("take one eager step() before capture(): it loads every kernel and driver entry point outside "
                               "the capture, and the first ab2 step (forward Euler, no H^{n-1}) is a different sequence")
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        graph = torch.cuda.CUDAGraph()
        n0 = self.launches
        with torch.cuda.graph(graph, stream=side):
            self.step(stream=torch.cuda.current_stream())
        torch.cuda.current_stream().wait_stream(side)
        self._graph, self._graph_launches = graph, self.launches - n0
        graph.replay()                              # capture does not execute: this is the step the call advances by
        return self

    def replay(self):
        """One time step through the captured graph."""
        if self._graph is None:
            raise RuntimeError("capture() first")
        self._graph.replay()
        self.steps += 1
        self.launches += self._graph_launches
