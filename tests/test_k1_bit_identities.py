"""Host-side checks (no GPU) of the two bit-level identities K1 v3 relies on, restated in plain Python
and compared with brute force: (1) the five-stage exchange network turns 8 words into their 8 bit planes in natural
byte order, and the boolean network over the planes equals the byte classes of include/driftsched.h; (2) two
carry-propagating adds over the continuation mask give every letter's position in its run mod 4."""
import random

M32 = 0xFFFFFFFF
WS_SET = {9, 10, 11, 12, 13, 32}


def _is_punct(c):
    return 0x21 <= c <= 0x2F or 0x3A <= c <= 0x40 or 0x5B <= c <= 0x60 or 0x7B <= c <= 0x7E


def _prmt(a, b, sel):
    pool = [(a >> (8 * i)) & 0xFF for i in range(4)] + [(b >> (8 * i)) & 0xFF for i in range(4)]
    return sum(pool[(sel >> (4 * i)) & 7] << (8 * i) for i in range(4))


def _exchange(a, b, s, m):
    return ((a & m) | ((b << s) & ~m)) & M32, (((a >> s) & m) | (b & ~m)) & M32


def _planes(w):
    w = list(w)
    for i in range(4):
        w[i], w[i + 4] = _prmt(w[i], w[i + 4], 0x5410), _prmt(w[i], w[i + 4], 0x7632)
    for i in (0, 1, 4, 5):
        w[i], w[i + 2] = _prmt(w[i], w[i + 2], 0x6240), _prmt(w[i], w[i + 2], 0x7351)
    for i in range(4):
        w[i], w[i + 4] = _exchange(w[i], w[i + 4], 2, 0x33333333)
    for i in (0, 1, 4, 5):
        w[i], w[i + 2] = _exchange(w[i], w[i + 2], 1, 0x55555555)
    for i in (0, 2, 4, 6):
        w[i], w[i + 1] = _exchange(w[i], w[i + 1], 4, 0x0F0F0F0F)
    return [w[0], w[2], w[4], w[6], w[1], w[3], w[5], w[7]]       # b0..b7 (register r holds plane k2=r&1, k1=r>>2, k0=r>>1&1)


def _classify(b):
    b0, b1, b2, b3, b4, b5, b6, b7 = b
    n = lambda x: ~x & M32
    mux = lambda sel, a, c: (sel & a) | (n(sel) & c)
    p15 = (n(b2) & (b1 | b0)) | (b2 & n(b1))
    p3 = b2 | (b1 & b0)
    p36 = b2 ^ (b1 & b0)
    pz = n(b2 | b1 | b0)
    g_even = n(b6) & (b5 | p15)
    g_odd = mux(b6, mux(b5, p36, p3), b5 & (b2 | b1))
    x = mux(b6, pz, b5)
    np_ = mux(b4, b3 & g_odd, mux(b3, g_even, x))
    letter = b7 | n(np_)
    q = n(b5) | (n(b3) & pz)
    ws = np_ & n(b6) & n(b4) & q & n(b7)
    return ws, letter


def test_transposition_and_class_network():
    rng = random.Random(1)
    for trial in range(600):
        by = [(trial * 32 + i) & 255 for i in range(32)] if trial < 8 else [rng.randrange(256) for _ in range(32)]
        w = [by[4 * i] | by[4 * i + 1] << 8 | by[4 * i + 2] << 16 | by[4 * i + 3] << 24 for i in range(8)]
        pl = _planes(w)
        for k in range(8):
            assert pl[k] == sum(((by[p] >> k) & 1) << p for p in range(32))
        ws, letter = _classify(pl)
        assert ws == sum((by[p] in WS_SET) << p for p in range(32))
        assert letter == sum((not (by[p] in WS_SET or _is_punct(by[p]))) << p for p in range(32))


W = 128
MW = (1 << W) - 1
_rep = lambda x: sum(x << (4 * i) for i in range(W // 4))


def _brute(L, S, carry_letter, cnt_in):
    f, cnt = 0, (cnt_in if carry_letter else 0)
    for p in range(W):
        if (S >> p) & 1:
            cnt = 0
        if (L >> p) & 1:
            if cnt % 4 == 0:
                f |= 1 << p
            cnt += 1
        else:
            cnt = 0
    return f


def _ripple(L, S, carry_letter, cnt_in):
    pl = ((L << 1) | (1 if carry_letter else 0)) & MW
    C = L & pl & ~S & MW
    first = C & ~((C << 1) & MW)
    r = (4 - cnt_in) & 3
    a_even, a_01 = first & _rep(0xA), first & _rep(0x6)
    if C & 1:
        a_even |= (r & 1) == 0
        a_01 |= r < 2
    s1, s2 = (C + a_even) & MW, (C + a_01) & MW
    u = C & ~(s1 ^ _rep(0xA)) & ~(s2 ^ _rep(0xC)) & MW
    return (u | (L & ~C)) & MW


def test_run_position_mod4_by_carry_ripple():
    rng = random.Random(5)
    for t in range(30000):
        mode = rng.random()
        if mode < 0.3:
            L = rng.getrandbits(W) | rng.getrandbits(W) | rng.getrandbits(W)
        elif mode < 0.6:
            L = rng.getrandbits(W)
        else:
            L = MW
            for _ in range(rng.randrange(4)):
                L &= ~(1 << rng.randrange(W))
        S = 0
        for _ in range(rng.randrange(5)):
            S |= 1 << rng.randrange(W)
        if rng.random() < 0.2:
            S |= 1
        carry, cnt = rng.random() < 0.6, rng.randrange(4)
        assert _brute(L, S, carry, cnt) == _ripple(L, S, carry, cnt)
