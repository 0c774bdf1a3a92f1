"""A CPU stand-in for the four hawkes_shard_* phases of HawkesContext, for the world-size-2 gloo test (tests only; the
product has no CPU path).  It evaluates exactly the pieces of the pair space that hawkes_plan_segments assigns to the
rank -- the cut is the library's own host code -- with the pair terms written out in numpy from Eq. 1 / Eq. 4
(readings R3 / R4 for the two indicators), at the log-likelihood level (want = LL | GRAD_THETA),
and forms the same partial-sum vectors the CUDA phases exchange.  `oracle/` is the judge of the assembled result."""
import numpy as np
import torch

import paper_2103_03348_b200 as hp

TILE = 256


class StubShardContext:
    def __init__(self, workers_per_rank: int = 5, symmetric: bool = True):
        self.W, self.sym = workers_per_rank, symmetric

    @staticmethod
    def shard_part_doubles(n, want, phase):
        return 2 * ((n + 255) // 256 * 256)

    def new_outputs(self, n, want):
        mk = lambda k: torch.zeros(k, dtype=torch.float64)
        return hp.EvalResult(ll=mk(1), grad_theta=mk(n))

    def _consts(self, params, dim):
        mu0, tx, tt, xi0, h, om = params
        cb = mu0 * (2 * np.pi) ** (-(dim + 1) / 2) * tx ** (-dim) / tt
        cs = xi0 * om * (2 * np.pi) ** (-dim / 2) * h ** (-dim)
        return cb, cs

    def _pairs(self, I, jb, je):
        n = self.t.shape[0]
        ti = np.arange(I * TILE, min(n, (I + 1) * TILE))
        sj = np.arange(jb, je)
        dx = self.x[:, ti][:, :, None] - self.x[:, sj][:, None, :]
        r2 = (dx * dx).sum(0)
        dt = self.t[ti][:, None] - self.t[sj][None, :]
        return ti, sj, r2, dt

    def shard_pass1(self, x, t, theta, params, want, rank, world, part_out):
        self.x, self.t, self.theta = x.numpy(), t.numpy(), theta.numpy()
        self.params = tuple(float(v) for v in params)
        n, dim = self.t.shape[0], self.x.shape[0]
        mu0, tx, tt, xi0, h, om = self.params
        cb, cs = self._consts(self.params, dim)
        ld = (n + 255) // 256 * 256
        b, s = np.zeros(ld), np.zeros(ld)
        for w, I, jb, je, slot in hp.plan_segments(n, 1, 0, self.sym, self.W * world, rank * self.W, (rank + 1) * self.W):
            ti, sj, r2, dt = self._pairs(I, jb, je)
            B = cb * np.exp(-r2 / (2 * tx * tx) - dt * dt / (2 * tt * tt)) * (r2 != 0)
            S = cs * self.theta[sj][None, :] * np.exp(-om * dt - r2 / (2 * h * h)) * (dt > 0)
            if self.sym:      # each unordered pair once: streamed index below the target's; B goes to both events
                once = sj[None, :] < ti[:, None]
                B = B * once
                S = S * once
                np.add.at(b, sj, B.sum(0))
            b[ti] += B.sum(1)
            s[ti] += S.sum(1)
        part_out[:ld] = torch.from_numpy(b)
        part_out[ld:] = torch.from_numpy(s)

    def shard_reduce1(self, n, params, want, world, parts_all, out):
        ld = (n + 255) // 256 * 256
        p = parts_all.numpy().reshape(world, 2, ld)
        lam = np.zeros(n)
        for r in range(world):                      # rank order
            lam += p[r, 0, :n] + p[r, 1, :n]
        self.lam = lam
        out.ll[0] = float(np.sum(np.log(lam)))      # the caller subtracts the integral term (the oracle's)

    def shard_pass2(self, n, params, want, rank, world, part2_out):
        dim = self.x.shape[0]
        mu0, tx, tt, xi0, h, om = self.params
        _, cs = self._consts(self.params, dim)
        ld = (n + 255) // 256 * 256
        c = np.zeros(ld)
        for w, M, jb, je, slot in hp.plan_segments(n, 2, 0, False, self.W * world, rank * self.W, (rank + 1) * self.W):
            si, tj, r2, dt = self._pairs(M, jb, je)   # sources of tile M (rows here), streamed targets [jb, je)
            dt = -dt                                   # t_target - t_source
            K = cs * np.exp(-om * dt - r2 / (2 * h * h)) * (dt > 0)
            c[si] += (K / self.lam[tj][None, :]).sum(1)
        part2_out[:ld] = torch.from_numpy(c)
        part2_out[ld:] = 0.0

    def shard_finish(self, n, params, want, world, parts2_all, out):
        ld = (n + 255) // 256 * 256
        p = parts2_all.numpy().reshape(world, 2, ld)
        c = np.zeros(n)
        for r in range(world):
            c += p[r, 0, :n]
        mu0, tx, tt, xi0, h, om = self.params
        out.grad_theta[:] = torch.from_numpy(c - xi0 * (-np.expm1(-om * (self.t[-1] - self.t))))
