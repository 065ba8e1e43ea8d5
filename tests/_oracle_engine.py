"""A CPU stand-in for ``paper_2606_19989_b200.dist.CudaEngine`` built from the ORACLE's pieces
(group_window, target_groups, align_list), used only by the world_size-2 gloo tests: it lets the
protocol driver of dist.py (the product's host-side logic: sequencing, collectives, termination on
the shared status) run on a box without a GPU.  Test infrastructure; never imported by the package."""
from types import SimpleNamespace

import numpy as np
import torch


class OracleEngine:
    def __init__(self, oracle, wl):
        self.o = oracle
        self.wl = wl
        self.p = wl.params
        self.params = SimpleNamespace(**wl.params)
        self.R = self.n_ranks = wl.n_ranks
        self.device = "cpu"
        self.fail_at_round = None      # tests: raise an engine error in form_groups of that round
        self.lens = [wl.lengths[wl.rank_ptr[r]:wl.rank_ptr[r + 1]] for r in range(self.R)]

    def local_max_window(self):
        m = max((len(x) for x in self.lens), default=0)
        bs = self.p["buffer_size"]
        return min(m, bs) if bs > 0 else m

    def dist_config(self, world_ranks, rank_offset, world_max_window):
        self.W, self.off = world_ranks, rank_offset
        bs, C = self.p["buffer_size"], self.p["slot_capacity"]
        b = world_max_window
        if C > 0:
            b = min(b, C)
        self.bound = max(b, 1)
        self.buf = [[] for _ in range(self.R)]
        self.pos = [0] * self.R
        self.slots = [[] for _ in range(self.R)]
        self.step_samples = []
        self.s_emit = 0
        self.round = 0
        self.stop = None
        self.world = torch.zeros(2 * world_ranks, dtype=torch.int32)
        self.local = torch.zeros(2 * self.R, dtype=torch.int32)
        self.arrived = None

    def set_available(self, h_arrived):
        self.arrived = None if h_arrived is None else [int(x) for x in h_arrived]

    def form_groups(self):
        if self.fail_at_round is not None and self.round == self.fail_at_round:
            from paper_2606_19989_b200 import binding as B
            raise B.OdbError(B.ODB_ERR_BAD_LENGTH, "OracleEngine.form_groups (injected failure)")
        bs = self.p["buffer_size"]
        self.cand = []
        for r in range(self.R):
            n_r = len(self.lens[r])
            lim = n_r if self.arrived is None else max(0, min(n_r, self.arrived[r]))
            while (bs == 0 or len(self.buf[r]) < bs) and self.pos[r] < lim:
                self.buf[r].append(self.pos[r])
                self.pos[r] += 1
            S = len(self.buf[r])
            g = self.o.group_window(self.p["rule"], self.p["budget"], self.lens[r], np.array(self.buf[r], np.int32)) if S else []
            self.cand.append(g)
            # S encoded as -1 when the rank is finished (nothing buffered, nothing pending), as k_pack_summary does
            self.local[2 * r], self.local[2 * r + 1] = len(g), (-1 if (S == 0 and self.pos[r] == n_r) else S)
        self.window = torch.zeros(self.bound, dtype=torch.int32)
        self.done = False
        self.T = 0

    def summary(self):
        return self.world, self.local

    def align(self):
        G, S = self.world[0::2].numpy().astype(np.int64), self.world[1::2].numpy().astype(np.int64)
        n_fin = int((S < 0).sum())
        self.done = (n_fin == self.W) if self.p["join_mode"] else (n_fin > 0)
        if self.done:
            return
        if not (G > 0).any():      # skip round: nobody has a group (all "insufficient data" or finished)
            self.T = 0
            self.aligned = [None] * self.R
            return
        self.T = self.o.target_groups(G, np.maximum(S, 0), self.p["slot_capacity"])
        self.aligned = []
        for r in range(self.R):
            if not self.cand[r]:
                self.aligned.append(None)
                continue
            al, back = self.o.align_list(self.cand[r], self.T)
            self.buf[r] = list(back)
            self.aligned.append(al)
            for k, g in enumerate(al):
                self.window[k] += len(g)

    def step_samples_window(self):
        return self.window

    def commit(self):
        if self.done:
            self.stop = 0 if self.p["join_mode"] else 1
            self.round += 1
            return
        e = self.window[:self.T].tolist()      # global after the all_reduce
        T_emit, Q = self.T, self.p["sample_quota"]
        if not self.p["join_mode"] and Q > 0:
            run = self.p["emitted_so_far"] + self.s_emit
            for k in range(self.T):
                run += e[k]
                if run >= Q:
                    T_emit = k + 1
                    self.stop = 2
                    break
        for r in range(self.R):
            for k in range(T_emit):
                self.slots[r].append(list(self.aligned[r][k]) if self.aligned[r] is not None else [])
            if self.aligned[r] is not None:
                for k in range(T_emit, self.T):
                    self.buf[r].extend(self.aligned[r][k])
        self.step_samples.extend(e[:T_emit])
        self.s_emit += sum(e[:T_emit])
        self.round += 1

    # ---- batched exchange (dist.py): every round that starts without leftovers, from the oracle's pieces ----
    def stream_lengths(self):
        return torch.tensor([len(x) for x in self.lens], dtype=torch.int32)

    def spec_form(self, n_rounds, world_max_stream):
        bs = self.p["buffer_size"]
        self.spec_J = n_rounds
        self.spec_cand = []
        g = torch.zeros(n_rounds * self.R, dtype=torch.int32)
        for j in range(n_rounds):
            row = []
            for r in range(self.R):
                ids = np.arange(min(j * bs, len(self.lens[r])), min((j + 1) * bs, len(self.lens[r])), dtype=np.int32)
                c = self.o.group_window(self.p["rule"], self.p["budget"], self.lens[r], ids) if len(ids) else []
                row.append(c)
                g[j * self.R + r] = len(c)
            self.spec_cand.append(row)
        self.spec_g = g
        self.window = torch.zeros(max(int(world_max_stream), 1), dtype=torch.int32)

    def spec_table(self):
        return self.spec_g

    def spec_commit(self, g_world, n_world, n_procs):
        bs, J = self.p["buffer_size"], self.spec_J
        G = g_world.numpy().astype(np.int64).reshape(n_procs, J, self.R)
        n = n_world.numpy().astype(np.int64).reshape(n_procs, self.R)
        self.spec_T, base = [], 0
        self.spec_sb = []
        for j in range(J):
            Gj = G[:, j, :].reshape(-1)
            Sj = np.clip(n.reshape(-1) - j * bs, 0, bs)
            if not (Gj > 0).any():
                break
            T = self.o.target_groups(Gj, Sj, self.p["slot_capacity"])
            if (Gj > T).any():      # some rank would overflow: leftovers, the round-by-round protocol takes over
                break
            self.spec_T.append(T)
            self.spec_sb.append(base)
            base += T
        for j, T in enumerate(self.spec_T):
            for r in range(self.R):
                cand = self.spec_cand[j][r]
                if cand:
                    al, back = self.o.align_list(cand, T)
                    assert len(back) == 0
                    for k, grp in enumerate(al):
                        self.window[self.spec_sb[j] + k] += len(grp)
                    self.slots[r].extend(list(x) for x in al)
                else:
                    self.slots[r].extend([] for _ in range(T))
        js = len(self.spec_T)
        for r in range(self.R):
            self.pos[r] = min(js * bs, len(self.lens[r]))
            self.buf[r] = []
        self.spec_steps = base

    def spec_step_window(self, n):
        return self.window[:n]

    def spec_status(self, max_rounds):
        e = self.window[:self.spec_steps].tolist()     # global after the all_reduce
        self.step_samples.extend(e)
        self.s_emit += sum(e)
        self.round = len(self.spec_T)
        done = len(self.spec_T) == self.spec_J
        if done:       # round J is the terminal check: counted, nothing emitted
            self.round += 1
            self.stop = 0 if self.p["join_mode"] else 1
        return len(self.spec_T), self.spec_steps, list(self.spec_T), int(done)

    def round_status(self):
        if self.done:
            return 1, 0
        return (1 if self.stop == 2 else 0), self.T

    def plan_query(self):
        return SimpleNamespace(n_rounds=self.round, n_steps=len(self.step_samples), stop_reason=self.stop,
                               slots=self.slots, step_samples=list(self.step_samples))
