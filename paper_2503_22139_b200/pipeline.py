"""One Stage-2/3 training step of PMF-STGR chained from the C-ABI operators:

    reference-frame Gaussians --gsvox_forward (C = 1)--> I_ref(x)                       Eq. 5
    MBC Gaussians, level i    --gsvox_forward (C = 3)--> e_{i,k}(x)                     Eq. 5
    e, w_{i,k}(p_b)           --gsvox_mbc_combine_forward--> d(x, p_b)                  Eq. 3
    I_ref, d                  --gsvox_warp_forward--> I(x, p_b) = I_ref(x + d(x, p_b))  Eq. 2
    I(., p_b), angle_b        --gsvox_project_forward--> DRR_b = P[I(x, p_b)]           Eq. 12, Eq. 6

and the same chain backwards from dL/dDRR to the gradients of every Gaussian parameter and of the
motion coefficients.  Orchestration only: every arithmetic step runs in the CUDA kernels of
libgsvox.so; this module allocates the intermediate device buffers once and passes pointers.
The CNN motion encoder, the losses and the optimiser of the paper are out of scope.
"""
import torch

from . import binding as B_


class Stage3Step:
    def __init__(self, grid, geom, n_ref, n_levels, batch, device="cuda"):
        """grid = (origin, spacing, dims) shared by I_ref, the MBC volumes and the DVFs; geom = cone-beam
        geometry dict; n_ref = number of reference Gaussians; n_levels = [n_1, n_2, ...] MBC Gaussians
        per level; batch = projections per step."""
        self.grid, self.geom, self.batch = grid, dict(geom), int(batch)
        self.dims = tuple(int(d) for d in grid[2])
        nx, ny, nz = self.dims
        self.L = len(n_levels)
        dev = torch.device(device)
        f = lambda *s: torch.empty(s, dtype=torch.float32, device=dev)
        self.plan_ref = B_.Plan(n_ref, grid, max_channels=1)
        self.plans = [B_.Plan(n, grid, max_channels=3) for n in n_levels]
        self.iref, self.e = f(1, nz, ny, nx), f(self.L, 3, nz, ny, nx)
        self.dvf, self.warped = f(batch, 3, nz, ny, nx), f(batch, nz, ny, nx)
        self.drr = f(batch, int(geom["nv"]), int(geom["nu"]))
        self.g_warped, self.g_dvf = f(batch, nz, ny, nx), f(batch, 3, nz, ny, nx)
        self.g_iref, self.g_e = f(1, nz, ny, nx), f(self.L, 3, nz, ny, nx)
        self.g_coef = f(batch, self.L, 3)
        # parameter gradients, allocated once: (d feat | d rho, d pos, d scale, d quat) per plan
        gset = lambda n, c: (f(n, c), f(n, 3), f(n, 3), f(n, 4))
        self.g_ref, self.g_levels = gset(n_ref, 1), [gset(n, 3) for n in n_levels]
        self.scratch = B_._project_scratch(B_.make_grid(*grid), batch, dev)
        self._saved = None
        # the four voxelizers are independent: each runs on its own stream so that the small binning kernels of one
        # overlap the brick kernels of another (the C ABI takes the stream; nothing else changes)
        self._side = [torch.cuda.Stream(device=dev) for _ in range(self.L)]

    def _fork(self):
        main = torch.cuda.current_stream()
        for st in self._side:
            st.wait_stream(main)
        return main

    def _join(self, main):
        for st in self._side:
            main.wait_stream(st)

    def fit(self, ref, levels, slack=1.05):
        """Size the (brick, Gaussian) key buffers for these Gaussians: preprocess once, read the device status
        (synchronises) and re-create any plan whose key capacity is too small.  Call once before the loop."""
        def fitted(plan, params, ch):
            plan.preprocess(*params[:3])
            st = plan.status()
            if st["overflow"]:
                plan = B_.Plan(plan.n_max, self.grid, max_channels=ch, key_capacity=int(slack * st["keys_needed"]) + 1024)
                plan.preprocess(*params[:3])
                assert not plan.status()["overflow"]
            return plan
        self.plan_ref = fitted(self.plan_ref, ref, 1)
        self.plans = [fitted(p, lv, 3) for p, lv in zip(self.plans, levels)]
        return self

    def forward(self, ref, levels, coef, angles):
        """ref = (pos, scale, quat, rho[n,1]); levels = [(pos, scale, quat, feat[n,3]), ...]; coef [B,L,3];
        angles: B radians (host).  -> drr [B, nv, nu] (a buffer owned by this object)."""
        main = self._fork()
        for i, lv in enumerate(levels):
            with torch.cuda.stream(self._side[i]):
                self.plans[i].preprocess(*lv[:3])
                self.plans[i].forward(lv[3], out=self.e[i])
        self.plan_ref.preprocess(*ref[:3])
        self.plan_ref.forward(ref[3], out=self.iref)
        self._join(main)
        B_.mbc_combine_forward(self.e, coef, out=self.dvf)
        B_.warp_forward(self.iref[0], self.dvf, self.grid, out=self.warped)
        B_.project_forward(self.warped, self.grid, self.geom, angles, out=self.drr, scratch=self.scratch)
        self._saved = (ref, levels, coef, list(angles))
        return self.drr

    def backward(self, grad_drr):
        """dL/dDRR [B,nv,nu] -> dict(ref=(d rho, d pos, d scale, d quat), levels=[(d feat, d pos, d scale, d quat)],
        coef=dL/dcoef [B,L,3]), buffers owned by this object (overwritten by the next call).  Must follow forward() of
        the same step."""
        ref, levels, coef, angles = self._saved
        B_.project_backward(grad_drr, self.grid, self.geom, angles, out=self.g_warped, scratch=self.scratch)
        B_.warp_backward(self.iref[0], self.dvf, self.grid, self.g_warped, grads=(self.g_iref[0], self.g_dvf))
        B_.mbc_combine_backward(self.e, coef, self.g_dvf, grads=(self.g_e, self.g_coef))
        main = self._fork()
        for i, lv in enumerate(levels):
            with torch.cuda.stream(self._side[i]):
                self.plans[i].backward(lv[3], self.g_e[i], grads=self.g_levels[i])
        self.plan_ref.backward(ref[3], self.g_iref, grads=self.g_ref)
        self._join(main)
        return {"ref": self.g_ref, "levels": self.g_levels, "coef": self.g_coef}
