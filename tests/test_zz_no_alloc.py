"""ds_tail_stats_static: the entry point that allocates nothing (its scratch is a fixed device array inside the library).

Collected LAST on purpose (file name): the suite runs with `pytest -x`, so a failure here hides no other test. The GPU test
depends on nothing the other tests leave behind (own seeded inputs, own output tensors) and on no earlier call of the entry
point: it passes alone in a fresh process and after the whole suite. Results are integers, so the bar is the one every
percentile test here uses: bit-exact, against the existing path (ds_tail_stats with a caller workspace).
"""
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_sources_never_allocate():
    # no cudaMalloc / cudaFree / host-allocating call anywhere in the CUDA sources: all memory is the caller's, or (for the
    # *_static entry point) a file-scope __device__ array whose address comes from cudaGetSymbolAddress
    csrc = os.path.join(ROOT, "paper_2606_02982_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        if f.endswith((".cu", ".cuh")):
            src = re.sub(r"//.*", "", open(os.path.join(csrc, f)).read())
            assert not re.search(r"\bcuda(Malloc\w*|Free\w*|HostAlloc|MallocAsync|FreeAsync)\s*\(", src), f
    ts = open(os.path.join(csrc, "tail_stats.cu")).read()
    assert "static __device__ __align__(256) unsigned char g_tail_scratch" in ts
    assert "cudaGetSymbolAddress((void**)&ptr, g_tail_scratch)" in ts


def _case(rng, n, n_seg, lo, hi, skip_frac=0.05, empty=()):
    v = rng.integers(lo, hi, n).astype(np.int64)
    s = rng.integers(0, n_seg, n).astype(np.int32)
    s[rng.random(n) < skip_frac] = -1                      # skipped values
    for e in empty:
        s[s == e] = -1                                     # an empty segment must come back as -1
    return v, s


@pytest.mark.gpu
def test_static_entry_point_matches_the_workspace_path_on_calls_in_a_row():
    import torch
    import paper_2606_02982_b200 as ds
    from paper_2606_02982_b200 import _lib
    dev = "cuda:0"
    rng = np.random.default_rng(20261105)
    cases = [
        # (values, seg ids, segments, percentiles): at the limit of 128 (segment, percentile) pairs, negative values too
        _case(rng, 300_000, 64, -5_000_000, 40_000_000) + (64, (50, 99)),
        # a small call right after it: 5 x 3 pairs, one empty segment, keys that differ in the low bits only
        _case(rng, 7_001, 5, 1_000_000, 1_000_256, empty=(3,)) + (5, (50, 95, 99)),
        # one segment, one percentile, a single value
        (np.array([42], np.int64), np.array([0], np.int32), 1, (50,)),
    ]
    cases.append(cases[0])                                  # and the first one again, over whatever the others left behind
    for v, s, n_seg, pct in cases:
        dv, dseg = torch.from_numpy(v).to(dev), torch.from_numpy(s).to(dev)
        want, wcnt = ds.tail_stats(dv, dseg, n_seg, pct)    # existing path: caller workspace
        out = torch.full((n_seg, len(pct)), -777, dtype=torch.int64, device=dev)
        cnt = torch.full((n_seg,), -777, dtype=torch.int64, device=dev)
        ds.tail_stats_static(dv, dseg, n_seg, out, cnt, pct)
        assert ds.device_status() == 0
        assert torch.equal(out, want) and torch.equal(cnt, wcnt), (n_seg, pct)
    # the empty segment of the second case reads -1 with count 0 (so the comparison above was not vacuous)
    v, s, n_seg, pct = cases[1]
    out = torch.empty((n_seg, len(pct)), dtype=torch.int64, device=dev)
    cnt = torch.empty((n_seg,), dtype=torch.int64, device=dev)
    ds.tail_stats_static(torch.from_numpy(v).to(dev), torch.from_numpy(s).to(dev), n_seg, out, cnt, pct)
    assert out[3].tolist() == [-1, -1, -1] and int(cnt[3]) == 0 and int(cnt.sum()) == int((s >= 0).sum())
    # beyond the built-in scratch: a clear error, nothing launched, outputs untouched
    v, s = _case(rng, 1000, 43, 0, 1000)
    out = torch.full((43, 3), -777, dtype=torch.int64, device=dev)
    cnt = torch.full((43,), -777, dtype=torch.int64, device=dev)
    n0 = ds.launch_count()
    for n_seg, pct in ((43, (50, 95, 99)), (129, (50,))):   # 129 pairs; 129 segments
        with pytest.raises(ds.DsError) as e:
            ds.tail_stats_static(torch.from_numpy(v).to(dev), torch.from_numpy(s).to(dev), n_seg, out, cnt, pct)
        assert e.value.code == _lib.DS_ELIMIT and "built-in scratch" in str(e.value)
    torch.cuda.synchronize()
    assert ds.launch_count() == n0 and bool((out == -777).all()) and bool((cnt == -777).all())
