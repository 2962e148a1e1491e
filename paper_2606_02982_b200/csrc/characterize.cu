// K1 — ds_characterize: single-pass HBM stream over packed prompt text (SURVEY.md §8(a) a1+a2).
//
// Definition (include/driftsched.h):
//   words[i]  = # maximal runs of non-WS bytes in prompt i
//   tokens[i] = # PUNCT bytes + sum over maximal LETTER runs of ceil(len/4)
// Per-byte flag form used here (equivalent):
//   wordstart[j] = nonWS[j] && (j starts a prompt || WS[j-1])
//   tokflag[j]   = PUNCT[j] || (LETTER[j] && (# letters before j in its run, runs reset at prompt starts) % 4 == 0)
//   words[i] = popcount(wordstart over [a,b)),  tokens[i] = popcount(tokflag over [a,b)).
//
// Design (v3, B200). The v2 kernel was bound by the ALU pipe (LOP3/SHF at half rate), not by HBM: 731 warp
// instructions per 2 KiB. v3 cuts that to about a third:
//  * every WARP is its own pipeline: it owns one contiguous span of 4 KiB chunks and a private stage (kStages = 1 since
//    r02: the refill is issued the moment the stage's bytes are in registers) filled by 2-D TMA tile copies (32 rows x
//    128 B, SWIZZLE_128B, one mbarrier per stage, issued by an elected lane): no block-wide barrier anywhere, and a lane
//    reads its own 128-byte row with eight conflict-free LDS.128;
//  * byte classification is BIT-SLICED: each 32-byte group (8 registers) is transposed into its 8 bit planes
//    (2 PRMT stages + 3 masked-shift stages, shifts issued as IMAD/IMAD.HI on the FMA pipe), after which WS and LETTER
//    are a ~20-LOP3 boolean network evaluated for 32 bytes at a time, and the results already are position masks;
//  * the mod-4 position inside a letter run comes from two carry-propagating ADDs (a start bit added to the run
//    ripples through it, so `L & ~(L + starts_of_class)` labels every byte of a run with the class of its start)
//    instead of a Kogge-Stone shift network;
//  * carries between lanes are one bit + one bit + a count mod 4 and compose associatively; carries between
//    chunks live in warp-uniform registers;
//  * prompt boundaries come from a 32-entry register window over offsets[], held as 32-bit positions relative to the
//    warp's span; the counts at a boundary are read back from a per-32-byte table {wordstart mask, token mask,
//    running count} that the owning lanes leave in the warp's shared-memory table `att`. A prompt that closes inside
//    the warp's span is a plain store, the (at most two) prompts cut by the span's edges are integer atomicAdds.
#include <cuda.h>

#include "common.cuh"

namespace ds {
namespace k1 {

// Launch shape (r02, measured on configs[2] at 8 GiB): ONE CTA of 24 warps per SM, one 4 KiB TMA stage per warp.
// The stage is refilled as soon as its bytes are in registers and a chunk's arithmetic (~575 warp instructions at 6 warps per
// scheduler) outlasts the refill's latency, so a second stage only costs shared memory: 9 KB per warp instead of 13 KB is what lets
// 24 warps (80 registers each, no spills) share an SM instead of 16. 8 warps x 2 CTAs x 2 stages: 4.61 TB/s; 16 x 1 x 2: 5.04;
// 12 x 2 x 1: 4.90; 20 x 1 x 1 (96 registers): 5.17; 24 x 1 x 1: 5.25; 25 x 1 x 1 (72 registers): 4.73; 32 x 1 x 1 with kSub = 1: 4.97.
#ifndef DS_K1_WARPS
#define DS_K1_WARPS 24
#endif
#ifndef DS_K1_STAGES
#define DS_K1_STAGES 1
#endif
#ifndef DS_K1_SUB
#define DS_K1_SUB 2
#endif
#ifndef DS_K1_CTAS
#define DS_K1_CTAS 1
#endif
constexpr int kWarps = DS_K1_WARPS;           // warps per CTA (each fully independent)
constexpr int kThreads = kWarps * 32;
constexpr int NW = 4;                         // 32-byte groups (= 32-bit mask words) per lane per chunk
constexpr int kSeg = 32 * NW;                 // 128 bytes per lane per chunk = one TMA box row
constexpr int kChunk = 32 * kSeg;             // 4 KiB per warp per step
constexpr int kStages = DS_K1_STAGES;         // TMA stages per warp
constexpr int kSub = DS_K1_SUB;               // chunks per boundary-attribution pass (amortises the window handling)
constexpr int kCtasPerSM = DS_K1_CTAS;
constexpr unsigned kFull = 0xffffffffu;
constexpr long long kInfOff = 0x7fffffffffffffffLL;
constexpr unsigned kNoRel = 0xffffffffu;      // "no boundary" in span-relative 32-bit positions
static_assert(kChunk % 4 == 0 && kSeg == 128, "a TMA box row is one 128-byte swizzle row");

struct Smem {
  alignas(1024) uint8_t data[kWarps][kStages][kChunk];   // SWIZZLE_128B needs 1024-byte aligned stages
  uint4 att[kWarps][kSub * kChunk / 32];                 // per 32-byte word: {wordstart mask, token mask, packed count before it}
  unsigned int sbits[kWarps][kSub * kChunk / 32];        // prompt-start bit per byte of the warp's current kSub chunks
  unsigned long long mbar[kWarps][kStages];
};

// ---- PTX wrappers: mbarrier + 2-D TMA tile copy (SASS: UTMALDG, SYNCS) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait_a(uint32_t bar, unsigned parity) {   // bar: shared-window address
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP_A:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra.uni WAIT_DONE_A;\n"
      "bra.uni WAIT_LOOP_A;\n"
      "WAIT_DONE_A:\n"
      "}\n" ::"r"(bar), "r"(parity)
      : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_LOOP:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra.uni WAIT_DONE;\n"
      "bra.uni WAIT_LOOP;\n"
      "WAIT_DONE:\n"
      "}\n" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// rows [row, row+32) x 128 bytes of the text viewed as u8[rows][128] -> 4 KiB at dst, 16-byte pieces XOR-swizzled by row&7
__device__ __forceinline__ void tma_load_rows(void* dst, const CUtensorMap* map, int row, unsigned long long* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                   smem_u32(dst)),
               "l"(map), "r"(0), "r"(row), "r"(smem_u32(bar))
               : "memory");
}

// ---- bit-sliced byte classification: 32 bytes (8 words) -> WS mask, LETTER mask ----
// Masked-shift exchange of one register-index bit with one position bit (distance S, M = positions keeping their
// register). The shifts are multiplies by run-time powers of two so that they issue on the FMA pipe (IMAD / IMAD.HI):
// the ALU pipe (LOP3, PRMT) is this kernel's limiter.
struct Mul { unsigned l1, l2, l4, r1, r2, r4, p16, n16; };   // 2, 4, 16, 2^31, 2^30, 2^28, 2^16, -2^16
__device__ __forceinline__ uint32_t shl_fma(uint32_t x, unsigned pow2) {
  uint32_t r;
  asm("mul.lo.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(pow2));
  return r;
}
__device__ __forceinline__ uint32_t shr_fma(uint32_t x, unsigned pow2_of_32_minus_s) {
  uint32_t r;
  asm("mul.hi.u32 %0, %1, %2;" : "=r"(r) : "r"(x), "r"(pow2_of_32_minus_s));
  return r;
}
template <uint32_t M>
__device__ __forceinline__ uint32_t bitsel(uint32_t x, uint32_t y) {   // (x & M) | (y & ~M) as ONE LOP3 with one immediate
  uint32_t r;
  asm("lop3.b32 %0, %1, %2, %3, 0xE4;" : "=r"(r) : "r"(x), "r"(y), "n"(M));
  return r;
}
template <uint32_t M>
__device__ __forceinline__ void exchange(uint32_t& a, uint32_t& b, unsigned ml, unsigned mr) {
  const uint32_t bs = shl_fma(b, ml), as = shr_fma(a, mr);
  a = bitsel<M>(a, bs);
  b = bitsel<M>(as, b);
}
__device__ __forceinline__ void prmt_pair(uint32_t& a, uint32_t& b, uint32_t s0, uint32_t s1) {
  const uint32_t x = __byte_perm(a, b, s0), y = __byte_perm(a, b, s1);
  a = x; b = y;
}
// 16-bit halves exchange [a.lo, b.lo] / [a.hi, b.hi] (PRMT 0x5410 / 0x7632) done with five multiply-adds instead of two
// PRMTs: five FMA-pipe slots are cheaper than two ALU-pipe slots here.
__device__ __forceinline__ uint32_t mad_fma(uint32_t x, unsigned m, uint32_t c) {
  uint32_t r;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(r) : "r"(x), "r"(m), "r"(c));
  return r;
}
__device__ __forceinline__ void halves_pair(uint32_t& a, uint32_t& b, const Mul& mu) {
  const uint32_t ah = shr_fma(a, mu.p16), bh = shr_fma(b, mu.p16);
  const uint32_t alo = mad_fma(ah, mu.n16, a);          // a - (a.hi << 16)
  a = mad_fma(b, mu.p16, alo);                          // (b << 16) + a.lo
  b = mad_fma(bh, mu.p16, ah);                          // (b.hi << 16) + a.hi
}
constexpr bool kHalvesOnFma = false;   // measured: no gain (an ALU-pipe op costs about two issue slots, an IMAD one)
// w[i] = bytes 4i..4i+3 of the group. Register index bits (a4,a3,a2), position bits (a1,a0 | k2,k1,k0); five exchanges
// bring the address bits into the position (natural byte order) and the bit index into the register index.
__device__ __forceinline__ void classify32(uint32_t (&w)[8], const Mul& mu, uint32_t& ws, uint32_t& letter) {
#pragma unroll
  for (int i = 0; i < 4; ++i) {                                                       // a4 <-> byte-index bit 1
    if (kHalvesOnFma) halves_pair(w[i], w[i + 4], mu); else prmt_pair(w[i], w[i + 4], 0x5410u, 0x7632u);
  }
#pragma unroll
  for (int i = 0; i < 8; ++i) if (!(i & 2)) prmt_pair(w[i], w[i + 2], 0x6240u, 0x7351u);   // a3 <-> byte-index bit 0
#pragma unroll
  for (int i = 0; i < 4; ++i) exchange<0x33333333u>(w[i], w[i + 4], mu.l2, mu.r2);    // -> position bit 1
#pragma unroll
  for (int i = 0; i < 8; ++i) if (!(i & 2)) exchange<0x55555555u>(w[i], w[i + 2], mu.l1, mu.r1);   // -> position bit 0
#pragma unroll
  for (int i = 0; i < 8; i += 2) exchange<0x0f0f0f0fu>(w[i], w[i + 1], mu.l4, mu.r4); // a2 <-> position bit 2
  // register r now holds bit plane k with k2 = r&1, k1 = (r>>2)&1, k0 = (r>>1)&1
  const uint32_t b0 = w[0], b4 = w[1], b1 = w[2], b5 = w[3], b2 = w[4], b6 = w[5], b3 = w[6], b7 = w[7];
  // Boolean network, written so that every line is one 3-input function (one LOP3): with m = (b2 b1 b0) the low nibble
  // is (b3, m), and per row r = (b6 b5 b4) the non-LETTER set is  b3 ? G_r(m) : H_r(m):
  //   r=0: G = m in 1..5 (9..13)   r=2: all 16          r=3: G = m >= 2 (58..63)   r=4,6: H = (m == 0) (64, 96)
  //   r=5: G = m >= 3 (91..95)     r=7: G = m in 3..6 (123..126)                    r=1: none;  bytes >= 0x80: none.
  const uint32_t p15 = (~b2 & (b1 | b0)) | (b2 & ~b1);      // m in 1..5
  const uint32_t p3 = b2 | (b1 & b0);                        // m >= 3
  const uint32_t p36 = b2 ^ (b1 & b0);                       // m in 3..6
  const uint32_t pz = ~(b2 | b1 | b0);                       // m == 0
  const uint32_t g_even = ~b6 & (b5 | p15);                  // G for rows 0, 2 (rows 4, 6: none)
  const uint32_t u = (b5 & p36) | (~b5 & p3);                // G for rows 7 / 5
  const uint32_t v = b5 & (b2 | b1);                         // G for row 3 (row 1: none)
  const uint32_t g_odd = (b6 & u) | (~b6 & v);
  const uint32_t x = (b6 & pz) | (~b6 & b5);                 // H for the rows with b4 = 0: rows 4, 6 / row 2
  const uint32_t y0 = (b3 & g_even) | (~b3 & x);             // rows with b4 = 0
  const uint32_t z = b3 & g_odd;                             // rows with b4 = 1 (H = none)
  const uint32_t np = (b4 & z) | (~b4 & y0);                 // non-LETTER among bytes < 0x80
  letter = b7 | ~np;
  const uint32_t q = ~b5 | (~b3 & pz);                       // within rows 0 and 2: all of row 0's, only 0x20 of row 2's
  const uint32_t t = np & ~b6 & ~b4;
  ws = t & q & ~b7;
}

__device__ __forceinline__ unsigned bfind(uint32_t x) {              // index of the most significant 1 bit, 0xffffffff for 0
  unsigned r;
  asm("bfind.u32 %0, %1;" : "=r"(r) : "r"(x));
  return r;
}
__device__ __forceinline__ bool is_ws_scalar(uint32_t c) { return (c - 9u) <= 4u || c == 32u; }
__device__ __forceinline__ bool is_letter_scalar(uint32_t c) {
  bool punct = (c - 0x21u) <= 0x0Eu || (c - 0x3Au) <= 6u || (c - 0x5Bu) <= 5u || (c - 0x7Bu) <= 3u;
  return !punct && !is_ws_scalar(c);
}

// s = a + b over NW 32-bit words (carry chain; the carry out of the top word is dropped)
__device__ __forceinline__ void add_wide(const uint32_t (&a)[NW], const uint32_t (&b)[NW], uint32_t (&s)[NW]) {
  static_assert(NW == 4, "carry chain written for four words");
  asm("add.cc.u32 %0, %4, %8;\n\t"
      "addc.cc.u32 %1, %5, %9;\n\t"
      "addc.cc.u32 %2, %6, %10;\n\t"
      "addc.u32 %3, %7, %11;"
      : "=r"(s[0]), "=r"(s[1]), "=r"(s[2]), "=r"(s[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]));
}

// Token flags of the lane's 128 bytes: PUNCT bytes, run starts, and continuation letters whose 0-based position in their
// run is a multiple of 4.
//   L = letter mask (bit p of word g = byte 32g+p), C = L & "previous byte is a letter" & ~prompt_start = letters that
//   CONTINUE a run (so prompt starts cut runs for free), r_in = position class of the virtual start of the run that
//   continues into bit 0 (= -count mod 4; used only if C bit 0 is set).
// A carry injected at the first continuation byte of a run ripples through the run's continuation bytes and clears
// them, so C & ~(C + inject_c) marks the runs whose START has a position class in set c; two adds (c = even, c in
// {0,1}) give both bits of the start's position mod 4, and a continuation byte is flagged iff its own position mod 4
// equals that.
__device__ __forceinline__ void token_flags(const uint32_t (&L)[NW], const uint32_t (&C)[NW], const uint32_t (&ws)[NW],
                                            unsigned r_in, uint32_t (&ft)[NW]) {
  uint32_t aE[NW], a01[NW], s1[NW], s2[NW];
#pragma unroll
  for (int g = 0; g < NW; ++g) {
    const uint32_t csh = __funnelshift_l(g ? C[g - 1] : 0u, C[g], 1);   // bit 0 of the lane: always a first continuation
    aE[g] = C[g] & ~csh & 0xAAAAAAAAu;                                  // start (= previous byte) at an even position
    a01[g] = C[g] & ~csh & 0x66666666u;                                 // start at a position = 0, 1 (mod 4)
  }
  const uint32_t c0 = C[0] & 1u;
  aE[0] |= c0 & ~r_in; a01[0] |= c0 & ~(r_in >> 1);
  add_wide(C, aE, s1); add_wide(C, a01, s2);
#pragma unroll
  for (int g = 0; g < NW; ++g) {
    const uint32_t t = C[g] & ~(s1[g] ^ 0xAAAAAAAAu);
    const uint32_t u = t & ~(s2[g] ^ 0xCCCCCCCCu);
    const uint32_t v = (L[g] & ~C[g]) | (~ws[g] & ~L[g]);              // run starts and PUNCT bytes
    ft[g] = u | v;
  }
}

// number of k in [0,n) with off[k] < pos; executed by one full warp, 32-ary search (offsets non-decreasing)
__device__ __forceinline__ long long warp_count_lt(const int64_t* __restrict__ off, long long n, long long pos, int lane) {
  long long lo = 0, hi = n;   // answer in [lo,hi]
  while (hi > lo) {
    const long long stride = (hi - lo + 31) / 32;
    const long long k = lo + (long long)lane * stride;         // probe k: is off[k] < pos ?
    const bool pred = (k < hi) && (off[k] < pos);
    const int c = __popc(__ballot_sync(kFull, pred));           // probes form a prefix
    if (c == 0) return lo;
    const long long last_true = lo + (long long)(c - 1) * stride;
    long long nhi = lo + (long long)c * stride;                 // first probe that failed (or beyond)
    if (nhi > hi) nhi = hi;
    lo = last_true + 1;
    hi = nhi;
  }
  return lo;
}

__global__ void __launch_bounds__(kThreads, kCtasPerSM)
characterize_kernel(const __grid_constant__ CUtensorMap tmap, const uint8_t* __restrict__ bytes, long long n_bytes,
                    const int64_t* __restrict__ off, long long n_prompts, int32_t* __restrict__ words, int32_t* __restrict__ tokens,
                    long long n_chunks, long long n_tma_chunks, unsigned int* status, Mul mu) {
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

  // the warp index through a warp reduction: its result lives in a uniform register, so everything derived from it (the
  // span, the TMA row and barrier operands) is uniform for the compiler and the TMA issue needs no operand-broadcast loop
  const int lane = threadIdx.x & 31, warp = (int)__reduce_max_sync(kFull, threadIdx.x >> 5);
  const long long gw = (long long)blockIdx.x * kWarps + warp, nw = (long long)gridDim.x * kWarps;
  const long long c_begin = gw * n_chunks / nw, c_end = (gw + 1) * n_chunks / nw;   // this warp's span of chunks
  if (c_begin >= c_end) return;                                                     // (no block-wide barrier below)

  const long long mis = (long long)((unsigned long long)bytes & 15ull);
  const uint8_t* abase = bytes - mis;                         // 16-byte aligned; chunk c = abase[c*kChunk, (c+1)*kChunk)
  const long long load_end = (mis + n_bytes + 15) & ~15ll;    // bytes from abase that may be read
  unsigned long long* mbar = sm.mbar[warp];
  uint8_t (*stage)[kChunk] = sm.data[warp];
  unsigned int* sb = sm.sbits[warp];

  if (lane == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&mbar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
#pragma unroll
  for (int k = 0; k < kSub * kChunk / 32 / 32; ++k) sb[lane + 32 * k] = 0u;
  __syncwarp();

  // chunks [0, n_tma_chunks) lie wholly inside the readable range and come by TMA; the last, partial one is read directly
  const unsigned n_it = (unsigned)(c_end - c_begin);
  const unsigned it_tma = n_tma_chunks <= c_begin ? 0u : (n_tma_chunks - c_begin >= (long long)n_it ? n_it : (unsigned)(n_tma_chunks - c_begin));
  const int row0 = (int)(c_begin * 32);   // first TMA row of the span (rows < 2^31: n_bytes <= 2^37 checked by the host)
  // shared-window addresses of the stages and their barriers, computed once (the generic->shared conversion per use costs
  // a dozen instructions in the loop)
  const uint32_t stage_a0 = smem_u32(stage[0]), mbar_a0 = smem_u32(&mbar[0]);
  auto issue = [&](unsigned it, int s) {  // one lane only
    if (it < it_tma) {
      const uint32_t bar = mbar_a0 + 8u * (unsigned)s, dst = stage_a0 + (unsigned)kChunk * (unsigned)s;
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"((unsigned)kChunk) : "memory");
      asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
                   "l"(&tmap), "r"(0), "r"(row0 + (int)it * 32), "r"(bar)
                   : "memory");
    }
  };
  if (lane == 0)
    for (unsigned it = 0; it < n_it && it < (unsigned)kStages; ++it) issue(it, (int)it);

  // ---- span prologue: boundary cursor and the carries at the span's first byte ----
  const long long nb_total = n_prompts + 1;                   // boundaries off[0..n_prompts]
  const long long pos0 = c_begin * (long long)kChunk - mis;   // position (relative to bytes) of the span's first byte
  long long kb = warp_count_lt(off, nb_total, pos0, lane);    // first boundary not before the span
  unsigned c_cnt = 0;                                         // letters (mod 4) of the run ending at pos0-1
  unsigned c_ws = 0x80000000u, c_L = 0u;                      // bit 31: byte pos0-1 is WS / is a LETTER (lane 0's carry-in)
  if (pos0 > 0) {
    const uint32_t pb = bytes[pos0 - 1];
    c_ws = is_ws_scalar(pb) ? 0x80000000u : 0u;
    c_L = is_letter_scalar(pb) ? 0x80000000u : 0u;
    const long long lb = kb >= 1 ? max((long long)off[kb - 1], 0ll) : 0ll;   // runs reset at the last boundary before pos0
    long long k = pos0 - 1;
    bool found = false;
    while (!found && k >= lb) {
      const long long j = k - lane;
      const bool brk = (j < lb) || !is_letter_scalar(bytes[j]);
      const unsigned m = __ballot_sync(kFull, brk);
      if (m) { c_cnt += __ffs(m) - 1; found = true; } else { c_cnt += 32; k -= 32; }
    }
    c_cnt &= 3u;
  }
  unsigned accW = 0, accT = 0;        // flags seen so far in the prompt that is open at the current position
  bool open_before_span = true;       // that prompt started before this warp's span (other warps add to it too)
  unsigned last_rel = 0;              // largest boundary seen, span-relative (validation of monotonicity across windows)

  // boundary window: lane holds off[kb + lane] as a 32-bit position relative to pos0 (kNoRel: none / beyond 4 GiB)
  unsigned orel = kNoRel;
  // per-lane cursors instead of 64-bit index arithmetic in the loop: this lane's entry of offsets[], how many entries are
  // left from it (<= 0: none), and the output slots of the prompt its boundary closes (boundary k closes prompt k-1)
  const int64_t* optr = off + kb + lane;
  long long left = nb_total - kb - lane;
  int32_t* wp = words + kb + lane - 1;
  int32_t* tp = tokens + kb + lane - 1;
  bool at_first = kb == 0;            // the window starts with boundary 0, which closes no prompt
  auto load_window = [&]() {
    const bool have = left > 0;
    const long long o = have ? *optr : kInfOff;
    const unsigned long long d = (unsigned long long)(o - pos0);
    orel = d >= (unsigned long long)kNoRel ? kNoRel : (unsigned)d;   // negative differences wrap to huge values
    unsigned prev = __shfl_up_sync(kFull, orel, 1);
    if (lane == 0) prev = last_rel;
    if (have && ((unsigned long long)o > (unsigned long long)n_bytes || o < pos0 || orel < prev)) atomicOr(status, DS_DEV_BAD_OFFSETS);
  };
  load_window();

  // lane's eight 16-byte pieces inside a stage (SWIZZLE_128B: piece p of row r sits at piece p ^ (r & 7))
  const uint8_t* lrow = &stage[0][0] + lane * kSeg;
  const unsigned lx = (unsigned)(lane & 7) << 4;
  const int lane_prev = (lane + 31) & 31;
  const unsigned lanemask_lt = (1u << lane) - 1u;
  unsigned scan_on[5];                  // 1 if lane >= 2^k: this lane takes the scan's k-th partial sum
#pragma unroll
  for (int k = 0; k < 5; ++k) {         // (asm volatile: keep them in registers instead of recomputing ISETP+SEL per chunk)
    const unsigned v = lane >= (1 << k) ? 1u : 0u;
    asm volatile("mov.u32 %0, %1;" : "=r"(scan_on[k]) : "r"(v));
  }

  // it_tail (32-bit, loop invariant) is the chunk that reaches past n_bytes
  const long long tail_chunk = (n_bytes + mis) / kChunk;      // first chunk whose end is beyond n_bytes
  const unsigned it_tail = tail_chunk < c_begin ? 0u : (tail_chunk - c_begin >= (long long)n_it ? kNoRel : (unsigned)(tail_chunk - c_begin));
  const bool head_edge = pos0 < 0;
  int s = 0;
  unsigned parity = 0, crel = 0;      // stage index, its mbarrier phase, chunk start relative to pos0
  uint4* att = sm.att[warp];
  for (unsigned it0 = 0; it0 < n_it; it0 += kSub, crel += kSub * kChunk) {   // kSub chunks: positions [pos0 + crel, +span)
  const unsigned nsub = n_it - it0 < (unsigned)kSub ? n_it - it0 : (unsigned)kSub;
  const unsigned span = nsub * (unsigned)kChunk;

  // (b) prompt boundaries inside these chunks -> start bits (the window's lanes hold them in order)
  unsigned rel = orel - crel;
  bool inb = rel < span;
  unsigned bm = __ballot_sync(kFull, inb);
  if (inb) atomicOr(&sb[rel >> 5], 1u << (rel & 31));
  if (bm == kFull) {                                     // rare: more than 32 boundaries may fall into the span
    const long long cs = pos0 + crel, ce = cs + span;
    const int64_t* o2p = optr;
    for (long long l2 = left - 32; ; l2 -= 32) {
      o2p += 32;
      if (__ballot_sync(kFull, l2 > 0) == 0u) break;
      const long long o2 = l2 > 0 ? *o2p : kInfOff;
      const bool in2 = o2 >= cs && o2 < ce;
      if (in2) atomicOr(&sb[(int)(o2 - cs) >> 5], 1u << ((int)(o2 - cs) & 31));
      if (__ballot_sync(kFull, in2) != kFull) break;
    }
  }
  __syncwarp();

  unsigned total = 0;                                    // packed count of the chunks of this pass so far
#pragma unroll
  for (unsigned h = 0; h < (unsigned)kSub; ++h) {
    if (h >= nsub) break;
    const unsigned it = it0 + h;
    const bool by_tma = it < it_tma;

    // (a) the lane's 128 bytes -> WS / LETTER masks, 32 bytes at a time
    uint32_t ws[NW], L[NW];
    if (by_tma) {
      mbar_wait_a(mbar_a0 + 8u * (unsigned)s, parity);
      const uint8_t* row = lrow + s * kChunk;
#pragma unroll
      for (int g = 0; g < NW; ++g) {
        const uint4 v0 = *reinterpret_cast<const uint4*>(row + (((2 * g) << 4) ^ lx));
        const uint4 v1 = *reinterpret_cast<const uint4*>(row + (((2 * g + 1) << 4) ^ lx));
        uint32_t w[8] = {v0.x, v0.y, v0.z, v0.w, v1.x, v1.y, v1.z, v1.w};
        classify32(w, mu, ws[g], L[g]);
      }
    } else {                            // partial last chunk: guarded 16-byte loads, zero beyond the readable range
      const long long a0 = (c_begin + it) * (long long)kChunk + lane * kSeg;
#pragma unroll
      for (int g = 0; g < NW; ++g) {
        uint4 v[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const long long a = a0 + (2 * g + h) * 16;
          v[h] = a < load_end ? *reinterpret_cast<const uint4*>(abase + a) : make_uint4(0u, 0u, 0u, 0u);
        }
        uint32_t w[8] = {v[0].x, v[0].y, v[0].z, v[0].w, v[1].x, v[1].y, v[1].z, v[1].w};
        classify32(w, mu, ws[g], L[g]);
      }
    }
    if ((head_edge && it == 0) || it >= it_tail) {   // cs < 0 or ce > n_bytes: bytes outside [0,n_bytes) count as whitespace
#pragma unroll
      for (int g = 0; g < NW; ++g) {
        const long long sp = pos0 + crel + (long long)(h * kChunk) + (long long)lane * kSeg + 32 * g;
        long long lo = -sp, hi = n_bytes - sp;
        lo = lo < 0 ? 0 : (lo > 32 ? 32 : lo);
        hi = hi < 0 ? 0 : (hi > 32 ? 32 : hi);
        uint32_t valid = 0u;
        if (hi > lo) valid = (hi == 32 ? ~0u : ((1u << hi) - 1u)) & ~((1u << lo) - 1u);
        ws[g] |= ~valid; L[g] &= valid;
      }
    }

    // the stage's bytes are all in registers now: refill it with the chunk kStages ahead
    __syncwarp();
    // One lane chosen by elect.sync issues the refill. With a `lane == 0` test the compiler wraps the (uniform-datapath) TMA
    // instruction in a vote-and-retry loop, 15 instructions per chunk; an elected lane needs none.
    if (it + kStages < it_tma) {
      unsigned elected;
      asm volatile("{\n.reg .pred p;\nelect.sync _|p, 0xffffffff;\nselp.u32 %0, 1, 0, p;\n}" : "=r"(elected));
      if (elected) issue(it + kStages, s);
    }
    const uint4 S4 = reinterpret_cast<const uint4*>(sb)[h * 32 + lane];
    reinterpret_cast<uint4*>(sb)[h * 32 + lane] = make_uint4(0u, 0u, 0u, 0u);
    const uint32_t S[NW] = {S4.x, S4.y, S4.z, S4.w};

    // (c) carries between lanes: one WS bit, one LETTER bit, the letter count (mod 4) of the run that is still open
    const unsigned rw = __shfl_sync(kFull, ws[NW - 1], lane_prev), rl = __shfl_sync(kFull, L[NW - 1], lane_prev);
    const unsigned wprev = lane ? rw : c_ws, lprev = lane ? rl : c_L;
    c_ws = rw; c_L = rl;                                              // lane 0 keeps lane 31's words for the next chunk
    uint32_t pw[NW], pl[NW];                                          // previous byte is WS / is a LETTER
#pragma unroll
    for (int g = 0; g < NW; ++g) {
      pw[g] = __funnelshift_l(g ? ws[g - 1] : wprev, ws[g], 1);
      pl[g] = __funnelshift_l(g ? L[g - 1] : lprev, L[g], 1);
    }
    uint32_t C[NW], call = ~0u;                                       // letters that continue a run; AND over the words
#pragma unroll
    for (int g = 0; g < NW; ++g) { C[g] = L[g] & pl[g] & ~S[g]; call &= C[g]; }
    const bool has_break = call != ~0u;
    // highest byte that does not continue its predecessor's run: the trailing run starts there (if a letter) or after it.
    // Common case: it lies in the top word. kz = number of trailing continuation bytes (mod 32; lower words add
    // multiples of 32 = 0 mod 4), the byte below them is bit 31-kz.
    uint32_t ct = C[NW - 1], lt = L[NW - 1];
    if (ct == ~0u && has_break) {                                    // rare: >= 32 trailing letters
      ct = C[2]; lt = L[2];
      if (ct == ~0u) { ct = C[1]; lt = L[1]; }
      if (ct == ~0u) { ct = C[0]; lt = L[0]; }
    }
    const unsigned hz = bfind(~ct);                                  // position of the highest 0 bit of ct
    const unsigned cnt_out = ((31u - hz) + ((lt >> (hz & 31u)) & 1u)) & 3u;   // garbage if !has_break: never read then
    const unsigned brk_mask = __ballot_sync(kFull, has_break);
    const unsigned below = brk_mask & lanemask_lt;
    const unsigned from_lane = __shfl_sync(kFull, cnt_out, bfind(below));      // bfind(0) = -1 -> lane 31, unused
    const unsigned cnt_in = below ? from_lane : c_cnt;
    const unsigned last_cnt = __shfl_sync(kFull, cnt_out, bfind(brk_mask));
    c_cnt = brk_mask ? last_cnt : c_cnt;                             // no break in the chunk: unchanged, 4096 = 0 (mod 4)

    // (d) flags and their counts per 32-byte word, packed words | tokens << 16
    uint32_t fw[NW], ft[NW], cpk[NW];
    token_flags(L, C, ws, (4u - cnt_in) & 3u, ft);
    unsigned own = 0;
#pragma unroll
    for (int g = 0; g < NW; ++g) {
      fw[g] = ~ws[g] & (S[g] | pw[g]);
      cpk[g] = (unsigned)__popc(fw[g]) + ((unsigned)__popc(ft[g]) << 16);
      own += cpk[g];
    }
    // table for the boundary pass: per 32-byte word {wordstart mask, token mask, packed count before the word}
    unsigned incl = own;                                              // inclusive prefix over lanes (0/1 multipliers: IMAD)
#pragma unroll
    for (int k = 0; k < 5; ++k) {
      const unsigned y = __shfl_up_sync(kFull, incl, 1 << k);
      asm("mad.lo.u32 %0, %1, %2, %0;" : "+r"(incl) : "r"(y), "r"(scan_on[k]));
    }
    unsigned run = total + incl - own;
#pragma unroll
    for (int g = 0; g < NW; ++g) { att[(h * 32 + lane) * NW + g] = make_uint4(fw[g], ft[g], run, 0u); run += cpk[g]; }
    total += __reduce_add_sync(kFull, own);                           // <= 8192 per field: no carry between the halves
    if (kStages == 2) { parity ^= (unsigned)s; s ^= 1; }             // the phase flips when the ring wraps from stage 1 to 0
    else if (++s == kStages) { s = 0; parity ^= 1u; }
  }
  __syncwarp();

  // (e) attribute to prompts: boundary k (= off[k]) closes prompt k-1
  {
    unsigned base_c = 0;                                              // packed prefix count at the last boundary handled
    if (bm) {
      for (;;) {
        const int nb = __popc(bm);
        const unsigned r = inb ? rel : 0u;
        const uint4 a = att[r >> 5];
        const unsigned mk = (1u << (r & 31)) - 1u;
        const unsigned cj = a.z + (unsigned)__popc(a.x & mk) + ((unsigned)__popc(a.y & mk) << 16);
        unsigned prev = __shfl_up_sync(kFull, cj, 1);
        if (lane == 0) prev = base_c;
        const unsigned dlt = cj - prev;                               // both fields are non-decreasing: no borrow
        unsigned nwd = dlt & 0xffffu, ntk = dlt >> 16;
        if (lane == 0) { nwd += accW; ntk += accT; }
        if (inb && !(at_first && lane == 0)) {                        // *wp / *tp: the prompt closed by this lane's boundary
          if (lane == 0 && open_before_span) {
            if (nwd) atomicAdd(wp, (int)nwd);
            if (ntk) atomicAdd(tp, (int)ntk);
          } else {
            *wp = (int)nwd; *tp = (int)ntk;
          }
        }
        accW = 0; accT = 0; open_before_span = false; at_first = false;
        base_c = __shfl_sync(kFull, cj, nb - 1);
        last_rel = __shfl_sync(kFull, orel, nb - 1);
        optr += nb; left -= nb; wp += nb; tp += nb;
        load_window();
        if (nb < 32) break;
        rel = orel - crel;
        inb = rel < span;
        bm = __ballot_sync(kFull, inb);
        if (!bm) break;
      }
    }
    const unsigned tail = total - base_c;
    accW += tail & 0xffffu; accT += tail >> 16;
    __syncwarp();
  }
  }

  // the prompt still open at the span's end continues in the next warp's span
  if (lane == 0 && !at_first && left > 0) {             // lane 0: next boundary kb with 1 <= kb <= n_prompts; wp = words + kb - 1
    if (accW) atomicAdd(wp, (int)accW);
    if (accT) atomicAdd(tp, (int)accT);
  }
}

}  // namespace k1

size_t ws_characterize(int64_t, int64_t) { return 256; }

}  // namespace ds

namespace {
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn encode_tiled() {   // driver entry point through the runtime: no link-time dependency on libcuda
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}
}  // namespace

extern "C" int ds_characterize(const uint8_t* bytes, int64_t n_bytes, const int64_t* offsets, int64_t n_prompts,
                               int32_t* words_out, int32_t* tokens_out, void* workspace, size_t workspace_bytes, void* stream) {
  using namespace ds;
  (void)workspace; (void)workspace_bytes;
  if (n_bytes < 0 || n_prompts < 0 || n_bytes > (1ll << 37)) return DS_EINVAL;   // 128 GiB: TMA row index stays below 2^31
  if (n_prompts > 0 && (!offsets || !words_out || !tokens_out)) return DS_EINVAL;
  if (n_bytes > 0 && !bytes) return DS_EINVAL;
  if (n_prompts == 0) return DS_OK;
  cudaStream_t st = (cudaStream_t)stream;
  unsigned int* status = status_ptr();
  if (!status) return cuda_fail(cudaGetLastError());
  DS_CUDA(cudaMemsetAsync(words_out, 0, sizeof(int32_t) * (size_t)n_prompts, st));
  DS_CUDA(cudaMemsetAsync(tokens_out, 0, sizeof(int32_t) * (size_t)n_prompts, st));
  if (n_bytes == 0) return DS_OK;
  const long long mis = (long long)((unsigned long long)bytes & 15ull);
  const long long load_end = (mis + n_bytes + 15) & ~15ll;
  const long long n_chunks = (mis + n_bytes + k1::kChunk - 1) / k1::kChunk;
  const long long n_tma_chunks = load_end / k1::kChunk;          // chunks wholly inside the readable range
  CUtensorMap tmap;
  memset(&tmap, 0, sizeof(tmap));
  if (n_tma_chunks > 0) {
    EncodeTiledFn enc = encode_tiled();
    if (!enc) return cuda_fail(cudaErrorNotSupported);
    const cuuint64_t dims[2] = {(cuuint64_t)k1::kSeg, (cuuint64_t)n_tma_chunks * 32ull};
    const cuuint64_t strides[1] = {(cuuint64_t)k1::kSeg};
    const cuuint32_t box[2] = {(cuuint32_t)k1::kSeg, 32u};
    const cuuint32_t estr[2] = {1u, 1u};
    if (enc(&tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, (void*)(bytes - mis), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
      return cuda_fail(cudaErrorInvalidValue);
  }
  if (attr_needed(DS_ATTR_K1))
    DS_CUDA(cudaFuncSetAttribute(k1::characterize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(k1::Smem)));
  long long grid = (long long)num_sms() * k1::kCtasPerSM;
  // small inputs: spread the chunks over CTAs as 8 per CTA rather than filling every warp of a few CTAs (a warp whose span is
  // empty returns at once), so that 1184 chunks (4.6 MiB) already reach every SM
  constexpr int kFill = k1::kWarps < 8 ? k1::kWarps : 8;
  const long long need = (n_chunks + kFill - 1) / kFill;
  if (grid > need) grid = need;
  const k1::Mul mu = {2u, 4u, 16u, 1u << 31, 1u << 30, 1u << 28, 1u << 16, 0u - (1u << 16)};
  k1::characterize_kernel<<<(unsigned)grid, k1::kThreads, sizeof(k1::Smem), st>>>(tmap, bytes, n_bytes, offsets, n_prompts, words_out,
                                                                               tokens_out, n_chunks, n_tma_chunks, status, mu);
  note_launch();
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}
