"""Pins for oracle.characterize: hand cases, Python bytes.split() (independent
library routine), an independent translate/split token reference, and the closed-form tokens/word ratio."""
import ast
import os
import re

import numpy as np
import pytest

import oracle
from paper_2606_02982_b200 import workload as wl


def _cases(golden_dir):
    out = []
    for line in open(os.path.join(golden_dir, "characterize_cases.txt")):
        if line.startswith("#") or not line.strip():
            continue
        lit, w, t = line.rstrip("\n").split("\t")
        out.append((ast.literal_eval(lit), int(w), int(t)))
    return out


def test_hand_cases(golden_dir):
    cases = _cases(golden_dir)
    assert len(cases) >= 12
    for s, w, t in cases:
        ow, ot = oracle.characterize(np.frombuffer(s, np.uint8), [0, len(s)])
        assert (int(ow[0]), int(ot[0])) == (w, t), s


def test_hand_cases_packed_neighbours(golden_dir):
    # a prompt edge always ends a word / run, whatever the neighbouring prompt holds
    cases = _cases(golden_dir)
    buf = b"".join(c[0] for c in cases)
    off = np.cumsum([0] + [len(c[0]) for c in cases])
    ow, ot = oracle.characterize(np.frombuffer(buf, np.uint8), off)
    assert ow.tolist() == [c[1] for c in cases]
    assert ot.tolist() == [c[2] for c in cases]
    # a word cut by a prompt boundary counts once per prompt
    ow, ot = oracle.characterize(np.frombuffer(b"abcdefgh", np.uint8), [0, 5, 8])
    assert ow.tolist() == [1, 1] and ot.tolist() == [2, 1]


_PUNCT = bytes(c for c in range(256) if chr(c) in r"""!"#$%&'()*+,-./:;<=>?@[\]^_`{|}~""")
_WS = b" \t\n\r\x0b\x0c"
_SPLIT_RE = re.compile(b"[" + re.escape(_WS + _PUNCT) + b"]+")


def _py_reference(buf: bytes, off):
    words, tokens = [], []
    for a, b in zip(off[:-1], off[1:]):
        s = buf[a:b]
        words.append(len(s.split()))                       # Python's own split(): PAPER.md:35
        n_punct = len(s) - len(s.translate(None, _PUNCT))   # punctuation bytes, counted by deletion
        tokens.append(n_punct + sum((len(p) + 3) // 4 for p in _SPLIT_RE.split(s) if p))
    return words, tokens


def test_against_python_split_random_bytes():
    rng = np.random.default_rng(7)
    # adversarial alphabet: every whitespace byte incl. 0x0b/0x0c/0x0d, near-misses (0x08,0x0e,0x1c-0x1f,0x85,0xa0),
    # punctuation range edges, letters, digits, high bytes
    alpha = np.frombuffer(b" \t\n\r\x0b\x0c\x08\x0e\x1c\x1f\x7f\x80\x85\xa0\xff!/:@[`{~09AZaz_\x00,.", np.uint8)
    buf = alpha[rng.integers(0, len(alpha), 6_000_000)]
    cuts = np.sort(rng.integers(0, buf.size + 1, 1_000_000))      # SURVEY.md §8(c) C.1 pin (1): >= 1 M prompts, WS runs of every length
    off = np.concatenate([[0], cuts, [buf.size]])
    w, t = oracle.characterize(buf, off)
    rw, rt = _py_reference(buf.tobytes(), off.tolist())
    assert w.tolist() == rw
    assert t.tolist() == rt


def test_against_python_split_scan_text():
    buf, off = wl.make_scan_text(2, 24 << 20)      # configs[2] generator: WS runs 0-8, edge runs, empty prompts
    w, t = oracle.characterize(buf, off)
    rw, rt = _py_reference(buf.tobytes(), off.tolist())
    assert w.tolist() == rw
    assert t.tolist() == rt
    assert (np.diff(off) == 0).sum() > 0


def test_all_256_byte_values_single():
    for c in range(256):
        s = bytes([c])
        w, t = oracle.characterize(np.frombuffer(s, np.uint8), [0, 1])
        ws = s in (b" ", b"\t", b"\n", b"\r", b"\x0b", b"\x0c")
        assert int(w[0]) == (0 if ws else 1)
        assert int(t[0]) == (0 if ws else 1)


@pytest.mark.parametrize("law,expect", [(wl.LAW0, 1.3977), (wl.LAW1, 2.1445)])
def test_closed_form_token_word_ratio(law, expect):
    # E[ceil(L/4)] = 1(1-q^4)+2(q^4-q^8)+3q^8 with L=min(12,Geom(p)), plus punctuation probability
    p, pp = law
    q = 1 - p
    closed = (1 - q**4) + 2 * (q**4 - q**8) + 3 * q**8 + pp
    assert abs(closed - expect) < 5e-4
    buf, off = wl.make_text(11, 4, 2000, law0=law)
    w, t = oracle.characterize(buf, off)
    assert abs(t.sum() / w.sum() - closed) < 0.004
    # generator words: 1-12 letters (+1 punct) -> word count equals the generator's draw range
    assert w.min() >= 5 and w.max() <= 200


def test_contract_violation():
    with pytest.raises(ValueError):
        oracle.characterize(np.zeros(4, np.uint8), [0, 5])
    with pytest.raises(ValueError):
        oracle.characterize(np.zeros(4, np.uint8), [3, 2])
