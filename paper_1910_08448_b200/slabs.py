"""1-D slab decomposition of one MPR problem over rows (include/mpr.h, "Slabs").

The grid of Ly rows is cut into G slabs of consecutive rows.  Slab i OWNS rows [own_begin, own_end) and holds, besides
them, `halo` rows of each neighbour (copies).  Every slab runs the ordinary kernels on all the rows it holds; a halo row
sees the slab's edge as an open boundary, so one colour pass spoils one more row from each inner edge: 4 rows per
hybrid sweep, 2 per quench double pass.  Before the spoiled region reaches the own rows -- every halo / 4 sweeps --
the halos are refreshed from their owners.  The random numbers are keyed on the GLOBAL site index (mpr_set_slab), so
the slabs together make, bit for bit, the moves of one context on the whole grid, for any G.

This module holds the host logic only: the partition, the order of sweeps and exchanges, and the two reductions a
measurement needs (the energy of a sweep is the sum of the slabs' parts; so is the sample energy).  It contains none
of the method's arithmetic.  `SlabSet` drives slab objects with the interface of `MprSlab` (a thin wrapper of
mpr.Mpr) through a transport:

  LocalTransport   every slab lives in this process (one GPU working the slabs off in turn -- how the GPU tests check
                   the decomposition against the single-context run -- or one process driving several GPUs);
  DistTransport    one slab per rank of a torch.distributed group: halo rows travel by send / recv (NCCL between GPUs
                   over NVLink; gloo with CPU staging in the CPU tests), energies by all_reduce.

On NVLink 5 / NVSwitch the exchange of a halo of 8 rows at L = 16384 is 2 x 8 x 64 KiB per neighbour and k = 2 sweeps:
latency-bound, which is why it is batched over k sweeps.
"""
from dataclasses import dataclass

import numpy as np


@dataclass(frozen=True)
class SlabPlan:
    index: int
    count: int
    rows: int            # Ly of the whole grid
    halo: int
    own_begin_g: int     # global rows this slab owns: [own_begin_g, own_end_g)
    own_end_g: int

    @property
    def row0_g(self):    # first global row the slab holds
        return self.own_begin_g - (self.halo if self.index > 0 else 0)

    @property
    def row1_g(self):    # one past the last global row it holds
        return self.own_end_g + (self.halo if self.index < self.count - 1 else 0)

    @property
    def n_rows(self):
        return self.row1_g - self.row0_g

    @property
    def own_begin(self):  # local
        return self.own_begin_g - self.row0_g

    @property
    def own_end(self):
        return self.own_end_g - self.row0_g


def plan_slabs(rows: int, count: int, halo: int):
    """Cuts `rows` rows into `count` slabs with a halo of `halo` rows.  halo is a multiple of 4 (whole hybrid sweeps
    between exchanges), every cut is at an even row (the colour of a site and the 2 x 2 quads of the float-mode random
    numbers are defined by the parity of the GLOBAL row) and every slab owns at least `halo` rows (a halo is filled by
    one neighbour)."""
    if count < 1 or halo < 4 or halo % 4:
        raise ValueError("count >= 1 and halo a positive multiple of 4")
    cuts = [0] + [(rows * i // count) // 2 * 2 for i in range(1, count)] + [rows]
    plans = []
    for i in range(count):
        if count > 1 and cuts[i + 1] - cuts[i] < halo:
            raise ValueError("%d rows are too few for %d slabs with a halo of %d" % (rows, count, halo))
        plans.append(SlabPlan(i, count, rows, halo, cuts[i], cuts[i + 1]))
    return plans


def bond_count(rows: int, cols: int) -> float:
    """Nearest-neighbour bonds of an open rows x cols grid (R3)."""
    return float(cols) * (rows - 1) + float(rows) * (cols - 1)


# ---- transports ----------------------------------------------------------------------------------------------------
class LocalTransport:
    """Every slab lives in this process."""
    rank = 0

    def owner(self, index):
        return 0

    def transfer(self, slabs, moves):
        """moves: (src slab, src row, dst slab, dst row, n rows).  All exports first, then all imports."""
        bufs = [slabs[src].export_rows(src_row, n) for (src, src_row, dst, dst_row, n) in moves]
        for buf, (src, src_row, dst, dst_row, n) in zip(bufs, moves):
            slabs[dst].import_rows(dst_row, n, buf)

    def reduce_sum(self, parts):
        return np.sum(np.stack([np.asarray(p, dtype=np.float64) for p in parts]), axis=0)

    def reduce_minmax(self, lo, hi):
        return float(min(lo)), float(max(hi))

    def gather_rows(self, plans, pieces):
        """pieces: {slab index: array of its own rows} -> the whole array (on every rank)."""
        return np.concatenate([pieces[p.index] for p in plans], axis=0)


class DistTransport:
    """One slab per rank of an initialised torch.distributed group (slab i on rank i)."""

    def __init__(self, group=None):
        import torch
        import torch.distributed as dist
        self._torch, self._dist, self.group = torch, dist, group
        self.rank = dist.get_rank(group)
        self.world = dist.get_world_size(group)
        self.cpu_staging = dist.get_backend(group) != "nccl"

    def owner(self, index):
        return index

    def _dev(self):
        return None if self.cpu_staging else self._torch.device("cuda", self._torch.cuda.current_device())

    def transfer(self, slabs, moves):
        torch, dist = self._torch, self._dist
        ops, recvs, keep = [], [], []
        for (src, src_row, dst, dst_row, n) in moves:
            if src == self.rank:
                buf = slabs[src].export_rows(src_row, n)
                if self.cpu_staging:
                    buf = buf.cpu()
                elif buf.is_cuda:
                    torch.cuda.current_stream(buf.device).synchronize()      # the export ran on the context's stream
                keep.append(buf)
                ops.append(dist.P2POp(dist.isend, buf, dst, self.group))
            if dst == self.rank:
                like = slabs[dst].rows_buffer(n)
                buf = like.cpu() if self.cpu_staging else like
                recvs.append((buf, like, dst_row, n))
                ops.append(dist.P2POp(dist.irecv, buf, src, self.group))
        if ops:
            for w in dist.batch_isend_irecv(ops):
                w.wait()
        for buf, like, dst_row, n in recvs:
            if self.cpu_staging:
                like.copy_(buf)
            slabs[self.rank].import_rows(dst_row, n, like)

    def reduce_sum(self, parts):
        t = self._torch.from_numpy(np.sum(np.stack([np.asarray(p, dtype=np.float64) for p in parts]), axis=0).copy())
        if self._dev() is not None:
            t = t.to(self._dev())
        self._dist.all_reduce(t, op=self._dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy()

    def reduce_minmax(self, lo, hi):
        t = self._torch.tensor([-min(lo), max(hi)], dtype=self._torch.float64)
        if self._dev() is not None:
            t = t.to(self._dev())
        self._dist.all_reduce(t, op=self._dist.ReduceOp.MAX, group=self.group)
        t = t.cpu()
        return -float(t[0]), float(t[1])

    def gather_rows(self, plans, pieces):
        mine = np.ascontiguousarray(pieces[self.rank])
        out = [None] * self.world
        self._dist.all_gather_object(out, mine, group=self.group)
        return np.concatenate(out, axis=0)


# ---- one slab on the CUDA path -------------------------------------------------------------------------------------
class MprSlab:
    """The rows plan.row0_g .. plan.row1_g of (values, mask) as an mpr.Mpr context in slab mode.  The interface SlabSet
    drives; tests/test_slabs_gloo.py drives the same SlabSet with a stand-in that needs no GPU."""

    def __init__(self, plan, values, mask, mode="DP", seed=0, device="cuda:0", path="AUTO", schedule="R4", stream=None):
        from . import mpr
        self.plan = plan
        self.stream = stream                 # a torch.cuda.Stream of this slab's own, or None (torch's current stream)
        v = np.ascontiguousarray(np.asarray(values)[plan.row0_g:plan.row1_g])
        m = np.ascontiguousarray(np.asarray(mask)[plan.row0_g:plan.row1_g])
        self.ctx = mpr.Mpr(v, m, mode=mode, seed=seed, device=device, slab=True, stream=stream)
        self.ctx.set_quench(0)              # SlabSet runs the quench passes itself, with halo refreshes in between
        self.ctx.set_path(path)
        self.ctx.set_schedule(schedule)
        self._mask_own = m[plan.own_begin:plan.own_end]
        self._values_own = v[plan.own_begin:plan.own_end]

    def local_range(self):
        """(z_min, z_max) of the measured values in the OWN rows."""
        z = self._values_own[self._mask_own == 0]
        return (float(z.min()), float(z.max())) if z.size else (float("inf"), float("-inf"))

    def configure(self, z_min, z_max, global_bonds):
        p = self.plan
        self.ctx.set_slab(p.row0_g, p.own_begin, p.own_end, z_min, z_max, global_bonds)

    def set_peers(self, up, down):
        self.ctx.set_peers(up.ctx if up is not None else None, down.ctx if down is not None else None)

    def sample_energy_parts(self):
        return self.ctx.sample_energy_parts()

    def n_free(self):
        return self.ctx.info()["n_free"]

    def set_temperature(self, T):
        self.ctx.set_temperature(T)

    def reset_chain(self, trial):
        self.ctx.reset_chain(trial)

    def quench(self, n_double_passes):
        self.ctx.quench(n_double_passes)

    def advance(self, n, measure=0, first_slot=0):
        self.ctx.advance(n, measure, first_slot)

    def fetch_series(self, n):
        return self.ctx.fetch_series(n)

    def accepted(self):
        return self.ctx.counters()[0]

    def rows_buffer(self, n):
        import torch
        return torch.empty(self.ctx.rows_bytes(n), dtype=torch.uint8, device=self.ctx.device)

    def export_rows(self, row, n):
        return self.ctx.export_rows(row, n)

    def import_rows(self, row, n, buf):
        self.ctx.import_rows(row, n, buf)

    def _done(self, t):
        if self.stream is not None:          # the kernel ran on this slab's stream, the copy below runs on torch's
            self.stream.synchronize()
        return t

    def own_state(self):
        p = self.plan
        return self._done(self.ctx.get_state())[p.own_begin:p.own_end].cpu().numpy()

    def own_prediction(self):
        p = self.plan
        return self._done(self.ctx.predict())[p.own_begin:p.own_end].cpu().numpy()


# ---- the orchestrator ----------------------------------------------------------------------------------------------
class SlabSet:
    """The slabs of one problem that live in this process (`slabs`: {index: slab}), driven in lock step.

    plans          plan_slabs(...) of the whole problem (every rank holds the same list)
    n_cols         Lx
    n_quench       quench double passes of a chain reset (R8), 32 in the library
    trial_lengths  (equilibration, measurement) sweeps of one temperature trial (R6): mpr.debug_trial_lengths()
    stats          series -> (mean, binned standard error), R16: mpr.debug_series_stats
    match          (e_sample, trial function T -> (e, se)) -> (T_hat, trial temperatures), R6: mpr.debug_match_temperature
    The last three are the library's own host routines (no GPU needed); they are arguments so that this module
    imports nothing of the method."""

    def __init__(self, plans, slabs, n_cols, transport, n_quench=32, trial_lengths=(200, 50), stats=None, match=None,
                 peer=False):
        self.plans, self.slabs, self.transport = plans, slabs, transport
        self.halo = plans[0].halo
        self.sweeps_per_exchange = self.halo // 4        # a hybrid sweep spoils 4 halo rows
        # peer mode (mpr_set_peers): every launch writes its edge rows straight into the neighbours' halos -- no exchange
        # step at all; needs all slabs in this process, a halo of 4 rows and an even number of quench double passes
        self.peer = bool(peer)
        if self.peer and (self.halo != 4 or len(slabs) != len(plans) or n_quench % 2):
            raise ValueError("peer mode: all slabs in one process, halo 4, even n_quench")
        self.n_cols = n_cols
        self.n_quench = n_quench
        self.trial_lengths = trial_lengths
        self._stats, self._match = stats, match
        self.T = None
        self.sweeps = 0
        self.n_trials = 0
        self.exchanges = 0
        # global range and bond count, then every slab is told its place
        lo, hi = zip(*[s.local_range() for s in slabs.values()])
        self.z_min, self.z_max = transport.reduce_minmax(lo, hi)
        self.bonds = bond_count(plans[0].rows, n_cols)
        for s in slabs.values():
            s.configure(self.z_min, self.z_max, self.bonds)
        parts = transport.reduce_sum([np.array(s.sample_energy_parts(), dtype=np.float64) for s in slabs.values()])
        self.n_pairs = int(round(parts[1]))
        self.e_sample = -2.0 * parts[0] / parts[1] if parts[1] > 0 else float("nan")
        self.n_free = int(round(transport.reduce_sum([np.array([s.n_free()], dtype=np.float64) for s in slabs.values()])[0]))
        if self.peer:
            for i, s in slabs.items():
                s.set_peers(slabs.get(i - 1), slabs.get(i + 1))
        # peer mode with a stream per slab: launch n + 1 of a slab waits for launch n of its neighbours (an event each)
        self._own_streams = self.peer and all(getattr(s, "stream", None) is not None for s in slabs.values())
        self._events = {}

    def moves(self):
        """The rows that travel in one refresh: every slab sends the `halo` own rows next to each inner edge."""
        out = []
        h = self.halo
        for p in self.plans[:-1]:
            q = self.plans[p.index + 1]
            out.append((p.index, p.own_end - h, q.index, q.own_begin - h, h))      # lower rows of p -> upper halo of q
            out.append((q.index, q.own_begin, p.index, p.own_end, h))              # upper rows of q -> lower halo of p
        return out

    def exchange(self):
        if len(self.plans) > 1 and not self.peer:
            self.transport.transfer(self.slabs, self.moves())
            self.exchanges += 1

    def _ordered(self, i, call):
        """Runs one launch round of slab i; with a stream per slab, after the neighbours' latest rounds."""
        if not self._own_streams:
            return call()
        import torch
        st = self.slabs[i].stream
        for j in (i - 1, i + 1):
            if j in self._events:
                st.wait_event(self._events[j])
        out = call()
        ev = torch.cuda.Event()
        ev.record(st)
        self._events[i] = ev
        return out

    def _barrier(self):
        if self._own_streams:
            import torch
            torch.cuda.synchronize()
            self._events = {}

    def set_temperature(self, T):
        self.T = float(T)
        for s in self.slabs.values():
            s.set_temperature(T)

    def reset_chain(self, trial=0):
        """R8: uniform spins (a function of the global site index and the trial: the halos agree without an exchange),
        then n_quench double passes; one double pass spoils 2 halo rows."""
        self._barrier()                       # the initialisation rewrites whole buffers, halos included
        for s in self.slabs.values():
            s.reset_chain(trial)
        self._barrier()
        per, done = self.halo // 2, 0
        while done < self.n_quench:
            m = min(per, self.n_quench - done)
            for i, s in self.slabs.items():
                self._ordered(i, lambda s=s: s.quench(m))
            self.exchange()
            done += m
        self.sweeps = 0

    def sweep(self, n):
        """n hybrid sweeps, halo / 4 at a time."""
        k = self.sweeps_per_exchange
        done = 0
        while done < n:
            m = min(k, n - done)
            for i, s in self.slabs.items():
                self._ordered(i, lambda s=s: s.advance(m, 0, 0))
            self.exchange()
            done += m
        self.sweeps += n

    def measure(self, n, accumulate):
        """n measuring sweeps -> the energy series of the whole grid (the sum of the slabs' parts)."""
        # one sweep per call (each has its own series slot); the halos last halo / 4 sweeps.  The energy of a sweep is
        # exact although the innermost halo row is then partly stale: a bond is counted at its colour-1 end, and the
        # colour-0 sites of that row -- the only halo sites an owned colour-1 site is bonded to -- go stale one pass later
        k = self.sweeps_per_exchange
        for i in range(n):
            for j, s in self.slabs.items():
                self._ordered(j, lambda s=s: s.advance(1, 2 if accumulate else 1, i))
            if (i + 1) % k == 0 or i + 1 == n:
                self.exchange()
        self.sweeps += n
        return self.transport.reduce_sum([s.fetch_series(n) for s in self.slabs.values()])

    def trial_energy(self, T):
        """One temperature trial of R6: a fresh chain keyed on the trial index, fixed sweep counts, energy only."""
        self.n_trials += 1
        self.set_temperature(T)
        self.reset_chain(self.n_trials)
        self.sweep(self.trial_lengths[0])
        series = self.measure(self.trial_lengths[1], accumulate=False)
        return self._stats(series)

    def estimate_temperature(self):
        """R6 on the whole grid: the library's root search, every trial run on all slabs.  Every rank sees the same
        (all-reduced) energies, so every rank takes the same decisions."""
        if not self.n_pairs:
            raise ValueError("no measured nearest-neighbour pair")
        self.n_trials = 0
        T_hat, _asked = self._match(self.e_sample, self.trial_energy)
        self.set_temperature(T_hat)
        self.reset_chain(0)
        return T_hat

    def run(self, n_eq, n_meas):
        """n_eq equilibration sweeps, n_meas measuring sweeps -> (energy series, mean, standard error).  The chain
        continues from where it is (reset_chain first for a fresh one), like mpr_run."""
        if self.T is None:
            raise ValueError("temperature not set")
        self.sweep(n_eq)
        series = self.measure(n_meas, accumulate=True)
        mean, se = self._stats(series) if n_meas else (float("nan"), 0.0)
        return series, mean, se

    def accepted(self):
        return int(round(self.transport.reduce_sum([np.array([s.accepted()], dtype=np.float64) for s in self.slabs.values()])[0]))

    def state(self):
        """phi of the whole grid (own rows of every slab, gathered on every rank)."""
        return self.transport.gather_rows(self.plans, {i: s.own_state() for i, s in self.slabs.items()})

    def prediction(self):
        return self.transport.gather_rows(self.plans, {i: s.own_prediction() for i, s in self.slabs.items()})


def make_slab_set(values, mask, count, halo=8, mode="DP", seed=0, device="cuda:0", path="AUTO", schedule="R4",
                  transport=None, n_quench=32, peer=False, streams=False):
    """The CUDA path on `count` slabs.  transport None: all slabs in this process on `device`; a DistTransport: this rank
    builds slab number transport.rank only (count = world size)."""
    from . import mpr
    mask = np.asarray(mask)
    plans = plan_slabs(int(mask.shape[0]), count, halo)
    transport = transport or LocalTransport()
    mine = [p for p in plans if transport.owner(p.index) == transport.rank]
    def own_stream():
        import torch
        return torch.cuda.Stream(device=device) if (peer and streams) else None
    slabs = {p.index: MprSlab(p, values, mask, mode=mode, seed=seed, device=device, path=path, schedule=schedule,
                              stream=own_stream()) for p in mine}
    return SlabSet(plans, slabs, int(mask.shape[1]), transport, n_quench=n_quench, trial_lengths=mpr.debug_trial_lengths(),
                   stats=mpr.debug_series_stats, match=mpr.debug_match_temperature, peer=peer)
