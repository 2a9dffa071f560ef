"""Host-side logic of the multi-GPU path: the hot path shards over independent windows
(gwi_infer) or over contiguous time spans of a stream (gwi_stream_*); models are replicated and no collective sits on
the data path (one rank per GPU, no inter-rank traffic during inference).  The only exchange is at the
end: timing (max over ranks), trigger counts, and -- for time shards -- the runs that touch a shard edge, which are
merged here.  No arithmetic of the network lives in this module; it is index bookkeeping, tested on CPU with gloo.
"""
from dataclasses import dataclass
from typing import List, Sequence, Tuple


def plan_windows(n_windows: int, world: int) -> List[Tuple[int, int]]:
    """Contiguous [start, end) window ranges, sizes differing by at most one, in rank order."""
    base, extra = divmod(int(n_windows), int(world))
    out, pos = [], 0
    for r in range(world):
        n = base + (1 if r < extra else 0)
        out.append((pos, pos + n))
        pos += n
    return out


@dataclass
class TimeShard:
    rank: int
    start: int          # first output sample this rank owns
    end: int            # one past the last
    warm_start: int     # first input sample it has to read: start - (R_f - 1), clipped at 0 (exact history, pin P8)
    l1_start: int       # first L1 sample it needs for the slides: warm_start - max_lag, clipped at 0 (the circular wrap
                        # of rank 0 is served by the stream tail, as in gwi_stream_prime)


def plan_time(n_samples: int, world: int, receptive_field: int, max_lag: int = 0, align: int = 1) -> List[TimeShard]:
    """Contiguous time spans, boundaries on multiples of `align`, each with the warm-up it needs in front."""
    out, pos = [], 0
    for r, (a, b) in enumerate(plan_windows((n_samples + align - 1) // align, world)):
        s, e = min(a * align, n_samples), min(b * align, n_samples)
        ws = max(0, s - (receptive_field - 1))
        out.append(TimeShard(r, s, e, ws, max(0, ws - max_lag)))
        pos = e
    assert pos == n_samples
    return out


def merge_shard_runs(shard_runs: Sequence[Sequence[Tuple[int, int]]], bounds: Sequence[Tuple[int, int]], min_len: int):
    """shard_runs[r]: ALL maximal supra-threshold runs [s, e) found inside shard r's span bounds[r] = (start, end), in
    global sample indices (min_len not yet applied; a run is cut at the span edges).  Runs that end exactly at a shard's
    end and a run that starts exactly at the next shard's start are one run of the whole stream.  Returns the merged
    runs of length >= min_len, sorted by start -- the list gwi_ensemble_triggers gives on the unsharded stream."""
    merged: List[List[int]] = []
    for r, runs in enumerate(shard_runs):
        lo, hi = bounds[r]
        for s, e in sorted(runs):
            assert lo <= s < e <= hi
            if merged and merged[-1][1] == s and s == lo and r > 0:
                merged[-1][1] = e           # continues the run that touched the previous shard's end
            else:
                merged.append([s, e])
    return [(s, e) for s, e in merged if e - s >= min_len]


def reduce_step_time(ms_local: float, dist=None) -> float:
    """Max over ranks of a per-rank device time (the bench contract); identity without a process group."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms_local)
    import torch
    t = torch.tensor([float(ms_local)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_objects(obj, dist=None):
    """All ranks' python objects on every rank (trigger lists / boundary runs are a few hundred bytes per rank)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [obj]
    out = [None] * dist.get_world_size()
    dist.all_gather_object(out, obj)
    return out


# ---- time shards through gwi_stream_* (include/gwi.h: gwi_stream_set_shard) --------------------------------------------
EDGE_LEFT, EDGE_RIGHT = 1 << 30, 1 << 29      # model_mask flags of a record that touches its shard's first / last sample


def shard_stream_args(n_global: int, start: int, end: int, receptive_field: int, max_lag: int = 0, align: int = 1):
    """What rank r, owner of the global samples [start, end), hands to gwi_stream_*:
    n_total (= warm-up + own samples), the shard tuple (t_first, warmup) of binding.Stream, the global index of its
    first pushed sample, and the global indices (circular) of the L1 samples it primes the slides with.  The warm-up is
    R_f - 1 samples rounded up to `align` (128 for the tensor-core slide back end), 0 for the owner of t = 0."""
    warm = 0 if start == 0 else -(-(receptive_field - 1) // align) * align
    warm = min(warm, start)
    first_pushed = start - warm
    n_total = end - first_pushed
    n_tail = max_lag + receptive_field - 1 if max_lag > 0 else 0     # gwi_stream_tail_samples() in shard mode
    tail_idx = [(first_pushed - n_tail + i) % n_global for i in range(n_tail)] if n_tail else []
    return {"n_total": n_total, "shard": (start, warm), "first_pushed": first_pushed, "tail_indices": tail_idx}


def merge_edge_records(records, min_len: int):
    """records: (slide, start, end, peak_p, mean_p, model_mask) of ALL shards, any order, as the shard-mode streams report
    them: runs >= min_len plus every run that touches a shard edge (flagged in model_mask).  A run flagged EDGE_RIGHT that
    ends where a run of the same slide flagged EDGE_LEFT starts is one run of the whole stream (chains over several shards
    join one after the other).  Returns the joined runs of length >= min_len sorted by (slide, start): the list the
    unsharded stream gives.  peak = max, mean = length-weighted, mask = OR of the parts (flags cleared)."""
    flags = EDGE_LEFT | EDGE_RIGHT
    out = []
    for slide, s, e, pk, mn, mask in sorted(records, key=lambda r: (r[0], r[1])):
        if out and out[-1][0] == slide and out[-1][2] == s and (out[-1][5] & EDGE_RIGHT) and (mask & EDGE_LEFT):
            p = out[-1]
            ln0, ln1 = p[2] - p[1], e - s
            p[2], p[3] = e, max(p[3], pk)
            p[4] = (p[4] * ln0 + mn * ln1) / (ln0 + ln1)
            p[5] = (p[5] & ~EDGE_RIGHT) | (mask & ~EDGE_LEFT)
        else:
            out.append([slide, s, e, pk, mn, mask])
    return [(r[0], r[1], r[2], r[3], r[4], r[5] & ~flags) for r in out if r[2] - r[1] >= min_len]
