"""A stand-in for paper_1910_08448_b200.slabs.MprSlab that needs no GPU: an integer cellular automaton with the SAME
dependency structure as the MPR sweep (checkerboard colours by the parity of the global coordinates, four colour passes
per sweep, each site rewritten from its own value and its four nearest neighbours, open boundaries -- also at the edge
of a slab, which is what spoils the halo rows) and none of its arithmetic.  Every quantity is an integer, so a slab run
must reproduce the whole-grid run EXACTLY, and any mistake in the host logic of slabs.py (partition, which rows travel,
how often, the order of exchange and measurement, the reductions) shows up as a mismatch.

The "spins" live in a torch CPU uint8 byte buffer when exported, like the real slab's rows."""
import numpy as np
import torch

MOD = 1 << 31


class ToySlab:
    def __init__(self, plan, values, mask, seed=0):
        self.plan = plan
        self.values = np.asarray(values)[plan.row0_g:plan.row1_g]
        self.mask = np.asarray(mask)[plan.row0_g:plan.row1_g].astype(bool)
        self.H, self.L = self.mask.shape
        self.seed = int(seed)
        self.T = 1.0
        self.state = np.zeros((self.H, self.L), dtype=np.int64)
        self.acc = np.zeros((self.H, self.L), dtype=np.int64)
        self.n_acc = 0
        self.series = np.zeros(4096)
        self.sweep_no = 0
        self._accepted = 0
        self.trial = 0
        yy, xx = np.mgrid[0:self.H, 0:self.L]
        self.gy = yy + plan.row0_g
        self.site = self.gy * self.L + xx                       # GLOBAL site index
        self.colour = (xx + self.gy) & 1
        self.own = (yy >= plan.own_begin) & (yy < plan.own_end)
        self.z_min = self.z_max = self.bonds = None

    # -- what SlabSet calls ------------------------------------------------------------------------------------------
    def local_range(self):
        z = self.values[self.own & ~self.mask]
        return (float(z.min()), float(z.max())) if z.size else (float("inf"), float("-inf"))

    def configure(self, z_min, z_max, bonds):
        self.z_min, self.z_max, self.bonds = z_min, z_max, bonds

    def sample_energy_parts(self):
        """pairs of measured sites to the right of and below the own rows; the toy 'cos' of every pair is 0.9"""
        m = ~self.mask
        right = m[:, :-1] & m[:, 1:] & self.own[:, :-1]
        down = m[:-1, :] & m[1:, :] & self.own[:-1, :]
        n = int(right.sum() + down.sum())
        return 0.9 * n, n

    def n_free(self):
        return int((self.mask & self.own).sum())

    def set_temperature(self, T):
        self.T = float(T)

    def reset_chain(self, trial):
        self.trial = int(trial)
        init = (self.site * 2654435761 + self.seed * 40503 + self.trial * 97) % MOD
        v = np.where(self.mask, self.z_min, self.values)                 # values at prediction sites are never used
        measured = np.floor((v - self.z_min) / (self.z_max - self.z_min) * 1000.0).astype(np.int64)
        self.state = np.where(self.mask, init, measured)
        self.acc[:] = 0
        self.n_acc = 0
        self.sweep_no = 0
        self._accepted = 0

    def _pass(self, colour, salt):
        s = self.state
        nb = np.zeros_like(s)
        nb[:, 1:] += s[:, :-1]
        nb[:, :-1] += s[:, 1:]
        nb[1:, :] += s[:-1, :]
        nb[:-1, :] += s[1:, :]
        new = (s * 1103515245 + nb * 12345 + self.site * 7 + salt) % MOD
        upd = self.mask & (self.colour == colour)
        self._accepted += int((upd & self.own & (new % 2 == 0)).sum())
        self.state = np.where(upd, new, s)

    def quench(self, n_double_passes):
        for _ in range(n_double_passes):
            self._pass(0, 11)
            self._pass(1, 11)

    def advance(self, n, measure=0, first_slot=0):
        for i in range(n):
            self.sweep_no += 1
            for k, colour in enumerate((0, 1, 0, 1)):
                self._pass(colour, 1000 * self.sweep_no + k + self.trial)
            if measure:
                # bonds counted at their colour-1 end, like the library: own colour-1 sites and their four neighbours
                s = self.state
                nb = np.zeros_like(s)
                nb[:, 1:] += s[:, :-1] % 1000
                nb[:, :-1] += s[:, 1:] % 1000
                nb[1:, :] += s[:-1, :] % 1000
                nb[:-1, :] += s[1:, :] % 1000
                part = int(((s % 1000 + nb) * ((self.colour == 1) & self.own)).sum())
                # monotone in T; the state-dependent part is a small integer multiple of 2^-40: sums of slabs are exact
                own_frac = float(self.own.sum()) / (self.plan.rows * self.L)
                self.series[first_slot + i] = (-2.0 + self.T) * own_frac + part * 2.0 ** -40
            if measure == 2:
                self.acc += self.state
                self.n_acc += 1

    def fetch_series(self, n):
        return self.series[:n].copy()

    def accepted(self):
        return self._accepted

    def rows_buffer(self, n):
        return torch.empty(n * self.L * 8, dtype=torch.uint8)

    def export_rows(self, row, n):
        return torch.from_numpy(np.ascontiguousarray(self.state[row:row + n]).view(np.uint8).reshape(-1).copy())

    def import_rows(self, row, n, buf):
        self.state[row:row + n] = buf.numpy().view(np.int64).reshape(n, self.L)

    def own_state(self):
        p = self.plan
        return self.state[p.own_begin:p.own_end].copy()

    def own_prediction(self):
        p = self.plan
        return self.acc[p.own_begin:p.own_end].copy()
