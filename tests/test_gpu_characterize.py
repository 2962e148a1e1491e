"""-m gpu: ds_characterize (through the C ABI) vs the oracle, element by element (bit-exact int32)."""
import ast
import os

import numpy as np
import pytest

pytestmark = pytest.mark.gpu

import oracle
from paper_2606_02982_b200 import workload as wl


@pytest.fixture(scope="module")
def G():
    import _gpuutil
    return _gpuutil


def _check(G, buf, off):
    ow, ot = oracle.characterize(buf, off)
    gw, gt = G.gpu_characterize(buf, off)
    assert np.array_equal(gw, ow), np.flatnonzero(gw != ow)[:10]
    assert np.array_equal(gt, ot), np.flatnonzero(gt != ot)[:10]


def test_hand_cases(G, golden_dir):
    cases = []
    for line in open(os.path.join(golden_dir, "characterize_cases.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lit, w, t = line.rstrip("\n").split("\t")
        cases.append((ast.literal_eval(lit), int(w), int(t)))
    buf = np.frombuffer(b"".join(c[0] for c in cases), np.uint8)
    off = np.cumsum([0] + [len(c[0]) for c in cases])
    gw, gt = G.gpu_characterize(buf, off)
    assert gw.tolist() == [c[1] for c in cases] and gt.tolist() == [c[2] for c in cases]


def test_all_byte_values(G):
    buf = np.arange(256, dtype=np.uint8)
    _check(G, buf, np.arange(257))
    _check(G, np.tile(buf, 300), np.arange(0, 256 * 300 + 1, 1))          # 76800 one-byte prompts
    _check(G, np.tile(buf, 300), np.array([0, 256 * 300]))               # one prompt, every byte pair class edge


def test_adversarial_random(G):
    rng = np.random.default_rng(7)
    alpha = np.frombuffer(b" \t\n\r\x0b\x0c\x08\x0e\x1c\x1f\x7f\x80\x85\xa0\xff!/:@[`{~09AZaz_\x00,.", np.uint8)
    buf = alpha[rng.integers(0, len(alpha), 3_000_000)]                   # ~183 tiles, ragged tail
    cuts = np.sort(rng.integers(0, buf.size + 1, 200_000))               # many empty / tiny prompts
    _check(G, buf, np.concatenate([[0], cuts, [buf.size]]))
    cuts = np.sort(rng.integers(0, buf.size + 1, 40))                    # prompts spanning many tiles
    _check(G, buf, np.concatenate([[0], cuts, [buf.size]]))
    _check(G, buf, np.concatenate([[1234], cuts[5:30], [buf.size - 777]]))  # bytes outside every prompt


def test_long_runs_and_carries(G):
    rng = np.random.default_rng(9)
    n = 1_200_000
    buf = np.full(n, ord("a"), np.uint8)                                 # one letter run across ~73 tiles
    _check(G, buf, np.array([0, n]))
    _check(G, buf, np.concatenate([[0], np.sort(rng.integers(0, n, 500)), [n]]))   # runs reset at prompt starts
    buf2 = buf.copy()
    buf2[rng.integers(0, n, 300)] = ord(",")
    buf2[rng.integers(0, n, 300)] = ord(" ")
    _check(G, buf2, np.concatenate([[0], np.sort(rng.integers(0, n, 500)), [n]]))
    for k in (1, 2, 3, 4, 5, 63, 64, 65, 16383, 16384, 16385):          # run lengths around the mod-4 / lane / tile seams
        b = np.full(40000, ord(" "), np.uint8)
        b[100:100 + k] = ord("x")
        b[16384 - 2:16384 - 2 + k] = ord("y")
        _check(G, b, np.array([0, 40000]))
        _check(G, b, np.array([0, 101, 16384, 16385, 40000]))


@pytest.mark.parametrize("mis", [1, 3, 8, 15])
def test_misaligned_base_pointer(G, mis):
    import torch
    import paper_2606_02982_b200 as ds
    buf, off = wl.make_scan_text(5, 1 << 20)
    big = torch.zeros(buf.size + 64, dtype=torch.uint8, device=G.DEV)
    big[mis:mis + buf.size] = torch.from_numpy(buf).to(G.DEV)
    view = big[mis:mis + buf.size]
    assert view.data_ptr() % 16 == mis
    w, t = ds.characterize(view, torch.from_numpy(off).to(G.DEV))
    ow, ot = oracle.characterize(buf, off)
    assert np.array_equal(w.cpu().numpy(), ow) and np.array_equal(t.cpu().numpy(), ot)


def test_scan_text_cfg2_scaled(G):
    buf, off = wl.make_scan_text(2, 96 << 20)                           # configs[2] generator, 6144 tiles
    _check(G, buf, off)


def test_cfg0_text(G):
    buf, off = wl.make_text(0, 1, 200)
    _check(G, buf, off)


def test_empty_inputs_and_bad_offsets(G):
    import torch
    import paper_2606_02982_b200 as ds
    w, t = G.gpu_characterize(np.zeros(0, np.uint8), np.zeros(5, np.int64))
    assert w.tolist() == [0] * 4 and t.tolist() == [0] * 4
    w, t = G.gpu_characterize(np.frombuffer(b"hello world", np.uint8), np.array([0], np.int64))
    assert w.size == 0
    text = torch.from_numpy(np.frombuffer(b"hello world, again", np.uint8).copy()).to(G.DEV)
    ds.characterize(text, torch.tensor([0, 12, 5, 18], dtype=torch.int64, device=G.DEV))
    assert ds.device_status() & 1                                        # DS_DEV_BAD_OFFSETS
    assert ds.device_status() == 0                                       # cleared by the read


def test_sizes_around_chunk_seams(G):
    # K1 v3 moves 4 KiB chunks by TMA (whole chunks only), reads the last partial chunk directly and handles boundaries
    # once per two chunks: buffer sizes and base misalignments around every one of those seams, dense and sparse prompts
    rng = np.random.default_rng(21)
    alpha = np.frombuffer(b"  \t\nabcdefghijklmnopqrstuvwxyz,.;", np.uint8)
    big = alpha[rng.integers(0, len(alpha), 3 * 8192 + 64)]
    for n in (1, 15, 16, 17, 4095, 4096, 4097, 8191, 8192, 8193, 12287, 12288, 12289, 16384, 3 * 8192 + 5):
        for mis in (0, 5):
            buf = big[mis:mis + n]
            dense = np.unique(np.concatenate([[0, n], rng.integers(0, n + 1, max(2, n // 3))]))
            sparse = np.unique(np.concatenate([[0, n], rng.integers(0, n + 1, 3)]))
            for off in (dense, sparse):
                w, k = G.gpu_characterize(buf, off) if mis == 0 else _misaligned(G, big, mis, n, off)
                ow, ok = oracle.characterize(buf, off)
                assert np.array_equal(w, ow) and np.array_equal(k, ok), (n, mis, len(off))


def _misaligned(G, big, mis, n, off):
    import torch
    import paper_2606_02982_b200 as ds
    t = torch.from_numpy(np.ascontiguousarray(big)).to(G.DEV)
    o = torch.from_numpy(np.ascontiguousarray(off, np.int64)).to(G.DEV)
    w, k = ds.characterize(t[mis:mis + n], o)
    assert ds.device_status() == 0
    return w.cpu().numpy(), k.cpu().numpy()
