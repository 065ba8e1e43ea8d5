"""Seeded synthetic workloads shaped like the paper's length distributions.

The paper's datasets (UltraChat-200K, LLaVA-150K, ShareGPT4o, MM-Mix;
PAPER.md:77, :183) are not available; these recipes stand in for them
(BASELINE.json `configs`, restated in DESIGN.md "Input recipe").  Everything
here is input generation only: lengths, masked spans, token ids.  No sorting,
grouping, alignment or collation happens in this module.

Draw order (so that any later session regenerates identical arrays): one
``numpy.random.default_rng(seed)`` per config; for r = 0..R-1 in order, whole
rank vectors are drawn as (i) text lengths, (ii) config-specific draws,
(iii) ``u`` for the prompt span.

Token ids are NOT drawn with numpy's generator; they are a pure integer hash of
the global token index (SplitMix64 finaliser), so a device can fill its own
input buffer and a host can regenerate any slice:

    tok[j] = ((mix64(seed * 0x9E3779B97F4A7C15 + j) >> 32) * VOCAB) >> 32
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence

import numpy as np

VOCAB = 151936
_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


# ----------------------------------------------------------------------------
# token ids (counter-based, pure integer)
# ----------------------------------------------------------------------------
def token_ids(seed: int, start: int, count: int) -> np.ndarray:
    """int32 token ids for global ragged-buffer indices [start, start+count)."""
    if count <= 0:
        return np.zeros(0, dtype=np.int32)
    out = np.empty(count, dtype=np.int32)
    chunk = 1 << 22
    with np.errstate(over="ignore"):
        base = np.uint64(seed) * _GOLDEN
        for c0 in range(0, count, chunk):
            c1 = min(count, c0 + chunk)
            z = np.arange(start + c0, start + c1, dtype=np.uint64) + base
            z ^= z >> np.uint64(30)
            z *= _M1
            z ^= z >> np.uint64(27)
            z *= _M2
            z ^= z >> np.uint64(31)
            hi = z >> np.uint64(32)
            out[c0:c1] = ((hi * np.uint64(VOCAB)) >> np.uint64(32)).astype(np.int32)
    return out


def tokens_for_samples(wl: "Workload", global_sample_ids: Sequence[int]):
    """Compact ragged token buffer holding only the listed samples.

    Returns (tokens int32, tok_off int64[len(ids)]) where sample k's tokens are
    tokens[tok_off[k] : tok_off[k] + length].  Used for sampled parity checks on
    workloads whose full token buffer is too large to hold on the host.
    """
    ids = np.asarray(global_sample_ids, dtype=np.int64)
    lens = wl.lengths[ids].astype(np.int64)
    off = np.zeros(len(ids), dtype=np.int64)
    if len(ids):
        off[1:] = np.cumsum(lens)[:-1]
    toks = np.empty(int(lens.sum()), dtype=np.int32)
    for k, g in enumerate(ids):
        toks[off[k]: off[k] + lens[k]] = token_ids(wl.token_seed, wl.token_start + int(wl.sample_ptr[g]), int(lens[k]))
    return toks, off


# ----------------------------------------------------------------------------
# workload container
# ----------------------------------------------------------------------------
@dataclass
class Workload:
    name: str
    n_ranks: int
    rank_ptr: np.ndarray      # int64 [R+1], rank-major sample ranges
    lengths: np.ndarray       # int32 [N]
    sample_ptr: np.ndarray    # int64 [N+1], token offsets into the ragged buffer
    span_ptr: np.ndarray      # int64 [N+1], CSR into span_lo/span_hi
    span_lo: np.ndarray       # int32, masked spans [lo,hi) in token positions
    span_hi: np.ndarray       # int32
    token_seed: int
    params: Dict[str, int] = field(default_factory=dict)
    token_start: int = 0      # global ragged-buffer index of this workload's first token (split_ranks)

    @property
    def n_samples(self) -> int:
        return int(self.rank_ptr[-1])

    @property
    def n_tokens(self) -> int:
        return int(self.sample_ptr[-1])

    def tokens(self) -> np.ndarray:
        """Full ragged int32 token buffer (only call when it fits in host RAM)."""
        return token_ids(self.token_seed, self.token_start, self.n_tokens)


_DEFAULT_PARAMS = dict(
    budget=2048, rule=0, join_mode=1, sample_quota=0, emitted_so_far=0,
    buffer_size=0, slot_capacity=0, pad_id=0, ignore_index=-100, shift_labels=1,
)


def _lognormal(rng, mean, cv, n):
    sigma2 = np.log(1.0 + cv * cv)
    mu = np.log(mean) - 0.5 * sigma2
    return rng.lognormal(mu, np.sqrt(sigma2), n)


def _assemble(name, per_rank_len, per_rank_spans, token_seed, params) -> Workload:
    """per_rank_spans[r] = (prompt_hi int64[n], vis_lo int64[n], vis_hi int64[n]); vis_lo==vis_hi -> none."""
    R = len(per_rank_len)
    rank_ptr = np.zeros(R + 1, dtype=np.int64)
    for r in range(R):
        rank_ptr[r + 1] = rank_ptr[r] + len(per_rank_len[r])
    if R:
        lengths = np.concatenate([np.asarray(x, dtype=np.int64) for x in per_rank_len]) if rank_ptr[-1] else np.zeros(0, np.int64)
    else:
        lengths = np.zeros(0, np.int64)
    N = int(rank_ptr[-1])
    sample_ptr = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(lengths, out=sample_ptr[1:])
    if N:
        p_hi = np.concatenate([s[0] for s in per_rank_spans]).astype(np.int64)
        v_lo = np.concatenate([s[1] for s in per_rank_spans]).astype(np.int64)
        v_hi = np.concatenate([s[2] for s in per_rank_spans]).astype(np.int64)
    else:
        p_hi = v_lo = v_hi = np.zeros(0, np.int64)
    has_p = p_hi > 0
    has_v = v_hi > v_lo
    # merge overlapping or touching spans so the CSR is sorted and disjoint
    merged = has_p & has_v & (p_hi >= v_lo)
    first_lo = np.where(has_p, 0, v_lo)
    first_hi = np.where(merged, np.maximum(p_hi, v_hi), np.where(has_p, p_hi, v_hi))
    n_sp = (has_p | has_v).astype(np.int64) + (has_p & has_v & ~merged).astype(np.int64)
    span_ptr = np.zeros(N + 1, dtype=np.int64)
    np.cumsum(n_sp, out=span_ptr[1:])
    span_lo = np.zeros(int(span_ptr[-1]), dtype=np.int32)
    span_hi = np.zeros(int(span_ptr[-1]), dtype=np.int32)
    one = n_sp >= 1
    span_lo[span_ptr[:-1][one]] = first_lo[one]
    span_hi[span_ptr[:-1][one]] = first_hi[one]
    two = n_sp == 2
    span_lo[span_ptr[:-1][two] + 1] = v_lo[two]
    span_hi[span_ptr[:-1][two] + 1] = v_hi[two]
    p = dict(_DEFAULT_PARAMS)
    p.update(params)
    return Workload(name, R, rank_ptr, lengths.astype(np.int32), sample_ptr, span_ptr,
                    span_lo, span_hi, int(token_seed), p)


def _prompt_only(rng, lens):
    u = rng.uniform(0.1, 0.5, len(lens))
    p_hi = np.floor(u * lens).astype(np.int64)
    z = np.zeros(len(lens), dtype=np.int64)
    return (p_hi, z, z)


# ----------------------------------------------------------------------------
# BASELINE.json configs (index 0..4)
# ----------------------------------------------------------------------------
def bj_config(index: int) -> dict:
    """Static description of BASELINE.json `configs[index]`."""
    table = [
        dict(name="tiny", R=2, n=64, budget=2048, seed=0),
        dict(name="lowcv_text", R=8, n=4096, budget=16384, seed=1),
        dict(name="multimodal", R=8, n=8192, budget=32768, seed=2),
        dict(name="highcv_longtail", R=16, n=16384, budget=65536, seed=3),
        dict(name="sweep", R=32, n=32768, budget=65536, seed=4),
    ]
    return dict(table[index])


def config5_cells():
    """The nine (CV, budget) cells of the throughput sweep, in a fixed order."""
    return [(cv, L) for cv in (0.3, 1.0, 2.5) for L in (16384, 65536, 262144)]


def make_workload(index: int, *, cv: Optional[float] = None, budget: Optional[int] = None,
                  rule: int = 0, join_mode: int = 1, n_ranks: Optional[int] = None,
                  n_per_rank: Optional[int] = None) -> Workload:
    """Build BASELINE.json config `index` (0-based).

    ``n_ranks`` / ``n_per_rank`` shrink a config for a bounded sample of the same
    distribution (first ranks / first samples of each rank are NOT a prefix of the
    full draw unless n_per_rank is left alone; use for timing samples only).
    Config 3 (index 3) in non-join mode gets the quota Q = R * floor(0.95 * min n_r).
    Config 4 (index 4) needs ``cv`` in {0.3, 1.0, 2.5}; the generator state is
    advanced through the earlier CVs so each CV's array is the documented one.
    """
    c = bj_config(index)
    R = c["R"] if n_ranks is None else n_ranks
    n = c["n"] if n_per_rank is None else n_per_rank
    L = c["budget"] if budget is None else budget
    rng = np.random.default_rng(c["seed"])
    lens_all: List[np.ndarray] = []
    spans_all = []
    params = dict(budget=L, rule=rule, join_mode=join_mode)
    name = c["name"]
    if index == 0:
        for _ in range(R):
            lens = rng.integers(8, 257, n).astype(np.int64)
            lens_all.append(lens)
            spans_all.append(_prompt_only(rng, lens))
    elif index == 1:
        for _ in range(R):
            lens = np.clip(np.rint(_lognormal(rng, 1024.0, 0.5, n)), 16, 8192).astype(np.int64)
            lens_all.append(lens)
            spans_all.append(_prompt_only(rng, lens))
    elif index == 2:
        for _ in range(R):
            text = np.maximum(np.rint(_lognormal(rng, 300.0, 0.8, n)), 1).astype(np.int64)
            has_img = rng.uniform(0.0, 1.0, n) < 0.7
            h28 = rng.integers(8, 49, n).astype(np.int64)
            w28 = rng.integers(8, 49, n).astype(np.int64)
            v = rng.uniform(0.0, 1.0, n)
            q = np.floor(v * (text + 1)).astype(np.int64)
            q = np.minimum(q, text)
            nv = np.where(has_img, h28 * w28, 0)
            lens = text + nv
            u = rng.uniform(0.1, 0.5, n)
            p_hi = np.floor(u * lens).astype(np.int64)
            lens_all.append(lens)
            spans_all.append((p_hi, q, q + nv))
    elif index == 3:
        for _ in range(R):
            body = _lognormal(rng, 512.0, 0.6, n)
            sel = rng.uniform(0.0, 1.0, n) < 0.1
            tail = 2048.0 * (1.0 + rng.pareto(1.2, n))
            lens = np.clip(np.rint(np.where(sel, tail, body)), 1, 32768).astype(np.int64)
            lens_all.append(lens)
            spans_all.append(_prompt_only(rng, lens))
        if not join_mode:
            params["sample_quota"] = R * int(np.floor(0.95 * n))
    elif index == 4:
        cvs = (0.3, 1.0, 2.5)
        if cv is None:
            cv = 1.0
        if cv not in cvs:
            raise ValueError("config 5 CV must be one of %r" % (cvs,))
        for this_cv in cvs:
            lens_all, spans_all = [], []
            for _ in range(R):
                lens = np.maximum(np.rint(_lognormal(rng, 2048.0, this_cv, n)), 1).astype(np.int64)
                lens_all.append(lens)
                spans_all.append(_prompt_only(rng, lens))
            if this_cv == cv:
                break
        name = "sweep_cv%g_L%d" % (cv, L)
    else:
        raise ValueError("config index must be 0..4")
    return _assemble(name, lens_all, spans_all, c["seed"], params)


# ----------------------------------------------------------------------------
# protocol test inputs (correctness only; SURVEY.md section 8(d) "Protocol tests")
# ----------------------------------------------------------------------------
def audit_distribution(kind: str, rng, n: int) -> np.ndarray:
    """The six 1000-sample audit distributions.

    Two of them print no ranges (reading U25): longtail = 90% U[32,256]
    + 10% U[1024,2048]; bimodal = 50% U[32,128] + 50% U[1024,2048].
    """
    if kind == "uniform_narrow":
        return rng.integers(64, 513, n)
    if kind == "uniform_wide":
        return rng.integers(64, 2049, n)
    if kind == "all_long":
        return rng.integers(1800, 2049, n)
    if kind == "all_short":
        return rng.integers(32, 65, n)
    if kind == "longtail":
        sel = rng.uniform(0, 1, n) < 0.1
        return np.where(sel, rng.integers(1024, 2049, n), rng.integers(32, 257, n))
    if kind == "bimodal":
        sel = rng.uniform(0, 1, n) < 0.5
        return np.where(sel, rng.integers(1024, 2049, n), rng.integers(32, 129, n))
    raise ValueError(kind)


AUDIT_KINDS = ("uniform_narrow", "uniform_wide", "longtail", "bimodal", "all_long", "all_short")


def protocol_workload(kind: str, seed: int = 0, **over) -> Workload:
    """Small multi-round inputs that fire overflow, IDLE slots, empty ranks and the quota cut."""
    rng = np.random.default_rng(1000 + seed)
    params: Dict[str, int] = {}
    if kind.startswith("audit:"):
        dist = kind.split(":", 1)[1]
        R = 8
        per = [audit_distribution(dist, rng, 125).astype(np.int64) for _ in range(R)]
        params = dict(budget=2048, buffer_size=128)
    elif kind == "overflow_multiround":
        R = 4
        per = [np.maximum(np.rint(_lognormal(rng, 256.0, 1.0, 512)), 1).astype(np.int64) for _ in range(R)]
        params = dict(budget=4096, buffer_size=64, slot_capacity=4)
    elif kind == "empty_rank":
        counts = list(range(47, 32, -1)) + [0]   # structure of PAPER.md Table 6 (:444)
        per = [rng.integers(8, 513, c).astype(np.int64) for c in counts]
        params = dict(budget=2048, buffer_size=16)
    elif kind == "unequal":
        per = [rng.integers(8, 513, c).astype(np.int64) for c in (1, 7, 300, 5000)]
        params = dict(budget=4096)
    elif kind == "fuzz":
        R = int(rng.integers(1, 6))
        per = [rng.integers(1, 65, int(rng.integers(0, 31))).astype(np.int64) for _ in range(R)]
        params = dict(budget=int(rng.choice([16, 64, 256])),
                      buffer_size=int(rng.choice([0, 1, 4, 16])),
                      slot_capacity=int(rng.choice([0, 1, 2, 5])),
                      rule=int(rng.integers(0, 2)),
                      join_mode=int(rng.integers(0, 2)),
                      shift_labels=int(rng.integers(0, 2)))
        if not params["join_mode"] and rng.uniform() < 0.5:
            tot = int(sum(len(p) for p in per))
            params["sample_quota"] = int(rng.integers(1, max(2, tot + 1)))
    else:
        raise ValueError(kind)
    params.update(over)
    spans = [_prompt_only(rng, p) for p in per]
    return _assemble(kind, per, spans, 7000 + seed, params)


def custom_workload(name: str, per_rank_lengths, seed: int = 0, **params) -> Workload:
    """A workload from explicit per-rank length arrays (prompt spans drawn with the usual rule)."""
    rng = np.random.default_rng(2000 + seed)
    per = [np.asarray(x, dtype=np.int64) for x in per_rank_lengths]
    spans = [_prompt_only(rng, p) for p in per]
    return _assemble(name, per, spans, 9000 + seed, params)


def offline_workload(n_ranks: int, seed: int = 0, *, n: int = 4096, mean: float = 512.0, cv: float = 1.0,
                     budget: int = 16384) -> Workload:
    """A GLOBAL pool of n samples for the offline comparators (F4: GMT / BMT / HFG): one
    length array for the whole job (rank_ptr = [0, n]) plus the random draws those planners consume, as inputs:
    ``perm`` (the epoch-seeded shuffle) and ``shuffle_key`` (one 31-bit key per potential batch)."""
    rng = np.random.default_rng(5000 + seed)
    lens = np.maximum(np.rint(_lognormal(rng, mean, cv, n)), 1).astype(np.int64)
    wl = _assemble("offline_pool", [lens], [_prompt_only(rng, lens)], 11000 + seed, dict(budget=budget, rule=1))
    wl.perm = rng.permutation(n).astype(np.int32)
    wl.shuffle_key = rng.integers(0, 2**31 - 1, max(n, 1)).astype(np.int32)
    wl.world = int(n_ranks)
    return wl


def split_ranks(wl: Workload, n_parts: int, bounds=None):
    """The same job held by ``n_parts`` processes: part p gets the consecutive ranks
    [p*R/n_parts, (p+1)*R/n_parts) with their samples, spans and (same hash indices) tokens.  Pure slicing.
    ``bounds`` (optional, n_parts + 1 rising rank indices from 0 to R) gives the processes unequal rank counts."""
    R = wl.n_ranks
    if bounds is None:
        assert R % n_parts == 0
        bounds = [p * (R // n_parts) for p in range(n_parts + 1)]
    assert len(bounds) == n_parts + 1 and bounds[0] == 0 and bounds[-1] == R
    parts = []
    for p in range(n_parts):
        r0, r1 = int(bounds[p]), int(bounds[p + 1])
        g0, g1 = int(wl.rank_ptr[r0]), int(wl.rank_ptr[r1])
        sp0, sp1 = int(wl.span_ptr[g0]), int(wl.span_ptr[g1])
        parts.append(Workload("%s[part %d/%d]" % (wl.name, p, n_parts), r1 - r0,
                              (wl.rank_ptr[r0:r1 + 1] - g0).copy(), wl.lengths[g0:g1].copy(),
                              (wl.sample_ptr[g0:g1 + 1] - wl.sample_ptr[g0]).copy(),
                              (wl.span_ptr[g0:g1 + 1] - sp0).copy(), wl.span_lo[sp0:sp1].copy(),
                              wl.span_hi[sp0:sp1].copy(), wl.token_seed, dict(wl.params),
                              wl.token_start + int(wl.sample_ptr[g0])))
    return parts


def describe(wl: Workload) -> dict:
    """Realised descriptors the paper uses for workloads: mean, CV, max, f_s."""
    l = wl.lengths.astype(np.float64)
    if len(l) == 0:
        return dict(n=0, mean=0.0, cv=0.0, max=0, f_s=0.0)
    mean = float(l.mean())
    return dict(n=int(len(l)), mean=mean, cv=float(l.std() / mean) if mean else 0.0,
                max=int(l.max()), f_s=float((l < wl.params["budget"] / 4.0).mean()),
                tokens=int(l.sum()))
