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
// Design (v2, B200): every WARP is its own pipeline. It owns one contiguous span of 2 KiB chunks and a private ring
// of kStages shared-memory stages filled by 1-D TMA bulk copies (cp.async.bulk + one mbarrier per stage, issued by
// lane 0), so there is no block-wide barrier anywhere and the LSU pipe carries no global loads of text. Each lane
// owns 64 contiguous bytes of the chunk: SWAR byte classification 4 bytes per 32-bit word (threshold adds on
// x|0x80808080, XOR-combined intervals, result masked to bit 7), bit-7 compaction by IDP4A with power-of-two
// weights, then pure 64-bit mask logic (Kogge-Stone stride-4 propagation for the mod-4 run position). Carries
// between lanes are 2 bits + 1 bit and compose associatively; carries between chunks live in warp-uniform registers.
// Prompt boundaries come from a 32-entry register window over offsets[]; a prompt that closes inside the warp's
// span is a plain store, the (at most two) prompts cut by the span's edges are integer atomicAdds.
#include "common.cuh"

namespace ds {
namespace k1 {

constexpr int kWarps = 8;                     // warps per CTA (each fully independent)
constexpr int kThreads = kWarps * 32;
constexpr int kSeg = 64;                      // bytes per lane per chunk
constexpr int kChunk = 32 * kSeg;             // 2 KiB per warp per step
constexpr int kStages = 4;
constexpr int kCtasPerSM = 3;
constexpr unsigned kFull = 0xffffffffu;
constexpr long long kInfOff = 0x7fffffffffffffffLL;

struct Smem {
  alignas(128) uint8_t data[kWarps][kStages][kChunk];
  unsigned long long mbar[kWarps][kStages];
  unsigned int sbits[kWarps][kChunk / 32];    // prompt-start bit per byte of the warp's current chunk
};

// ---- PTX wrappers: mbarrier + 1-D TMA bulk copy (SASS: UBLKCP, SYNCS) ----
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
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
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, unsigned bytes, unsigned long long* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst)),
               "l"(src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---- byte classification, 4 bytes per 32-bit word ----
// z = x|0x80808080 keeps every byte >= 0x80 so the per-byte subtractions never borrow across bytes; bit 7 of
// (z - n*0x01010101) is (low7(x) >= n). Intervals are XORs of nested thresholds. m = ~x & 0x80808080 both drops
// bytes >= 0x80 (LETTER) and clears the 7 low garbage bits, so the results are exactly 0x80 / 0x00 per byte.
// The threshold adds are issued as IMAD (z * one + (-n)) with a run-time `one` == 1 so that they execute on the FMA
// pipe: the ALU pipe (LOP3/SHF/ISETP, half rate) is the limiter of this kernel, not HBM.
__device__ __forceinline__ uint32_t thr(uint32_t z, uint32_t one, uint32_t n) {
  uint32_t t;
  asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(t) : "r"(z), "r"(one), "r"(0u - n * 0x01010101u));
  return t;
}
__device__ __forceinline__ uint32_t lop3_xor3(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ uint32_t lop3_xor_and(uint32_t a, uint32_t b, uint32_t c) {   // (a ^ b) & c
  uint32_t r;
  asm("lop3.b32 %0, %1, %2, %3, 0x28;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ void classify4(uint32_t x, uint32_t one, uint32_t& ws7, uint32_t& d7) {
  const uint32_t z = x | 0x80808080u;
  const uint32_t m = ~x & 0x80808080u;
  const uint32_t t9 = thr(z, one, 9), t14 = thr(z, one, 14), t32 = thr(z, one, 32), t33 = thr(z, one, 33);
  const uint32_t t48 = thr(z, one, 48), t58 = thr(z, one, 58), t65 = thr(z, one, 65), t91 = thr(z, one, 91);
  const uint32_t t97 = thr(z, one, 97), t123 = thr(z, one, 123), t127 = thr(z, one, 127);
  const uint32_t s1 = lop3_xor3(t9, t14, t32);              // [9,13] u [32,..)
  ws7 = lop3_xor_and(s1, t33, m);                           // WS = [9,13] u {32}
  const uint32_t a = lop3_xor3(t48, t58, t65), b = lop3_xor3(t91, t97, t123);
  d7 = lop3_xor_and(lop3_xor3(s1, a, b), t127, m);          // non-LETTER = WS u PUNCT
}

// 8 bytes holding 0x80/0x00 -> 128 * (8-bit mask): two IDP4A with weights 1,2,4,8 | 16,32,64,128
__device__ __forceinline__ uint32_t mask8x128(uint32_t w0, uint32_t w1) {
  uint32_t acc;
  asm("dp4a.u32.u32 %0, %1, %2, %3;" : "=r"(acc) : "r"(w0), "r"(0x08040201u), "r"(0u));
  asm("dp4a.u32.u32 %0, %1, %2, %3;" : "=r"(acc) : "r"(w1), "r"(0x80402010u), "r"(acc));
  return acc;
}

__device__ __forceinline__ bool is_ws_scalar(uint32_t c) { return (c - 9u) <= 4u || c == 32u; }
__device__ __forceinline__ bool is_letter_scalar(uint32_t c) {
  bool punct = (c - 0x21u) <= 0x0Eu || (c - 0x3Au) <= 6u || (c - 0x5Bu) <= 5u || (c - 0x7Bu) <= 3u;
  return !punct && !is_ws_scalar(c);
}

__device__ __forceinline__ int clz64(unsigned long long v) { return __clzll((long long)v); }
__device__ __forceinline__ unsigned long long shfl64(unsigned long long v, int src) {
  const unsigned lo = __shfl_sync(kFull, (unsigned)v, src), hi = __shfl_sync(kFull, (unsigned)(v >> 32), src);
  return ((unsigned long long)hi << 32) | lo;
}
// rotate left by 16*r bits, r in 0..3
__device__ __forceinline__ unsigned long long rotl16(uint32_t lo, uint32_t hi, int r) {
  const uint32_t a = (r & 2) ? hi : lo, b = (r & 2) ? lo : hi;          // after the 32-bit part of the rotation: (b:a)
  const int s = (r & 1) * 16;
  const uint32_t nlo = __funnelshift_l(b, a, s), nhi = __funnelshift_l(a, b, s);
  return ((unsigned long long)nhi << 32) | nlo;
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
characterize_kernel(const uint8_t* __restrict__ bytes, long long n_bytes, const int64_t* __restrict__ off, long long n_prompts,
                    int32_t* __restrict__ words, int32_t* __restrict__ tokens, long long n_chunks, unsigned int* status, unsigned int one) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);

  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long gw = (long long)blockIdx.x * kWarps + warp, nw = (long long)gridDim.x * kWarps;
  const long long c_begin = gw * n_chunks / nw, c_end = (gw + 1) * n_chunks / nw;   // this warp's span of chunks
  if (c_begin >= c_end) return;                                                     // (no block-wide barrier below)

  const long long mis = (long long)((unsigned long long)bytes & 15ull);
  const uint8_t* abase = bytes - mis;                         // 16-byte aligned
  const long long load_end = (mis + n_bytes + 15) & ~15ll;    // bytes from abase that may be read
  unsigned long long* mbar = sm.mbar[warp];
  uint8_t (*stage)[kChunk] = sm.data[warp];
  unsigned int* sb = sm.sbits[warp];

  if (lane == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&mbar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  sb[lane] = 0u; sb[lane + 32] = 0u;
  __syncwarp();

  auto issue = [&](unsigned it) {  // lane 0 only: chunk c_begin + it -> stage it % kStages
    const int s = (int)(it & (kStages - 1));
    const long long a0 = (c_begin + it) * (long long)kChunk;
    long long len = load_end - a0;
    if (len > kChunk) len = kChunk;
    mbar_expect_tx(&mbar[s], (unsigned)len);
    tma_load_1d(stage[s], abase + a0, (unsigned)len, &mbar[s]);
  };
  const unsigned n_it = (unsigned)(c_end - c_begin);
  if (lane == 0)
    for (unsigned it = 0; it < n_it && it < (unsigned)kStages; ++it) issue(it);

  // ---- span prologue: boundary cursor and the carries at the span's first byte ----
  const long long nb_total = n_prompts + 1;                   // boundaries off[0..n_prompts]
  const long long pos0 = c_begin * (long long)kChunk - mis;   // position (relative to bytes) of the span's first byte
  long long kb = warp_count_lt(off, nb_total, pos0, lane);    // first boundary not before the span
  unsigned c_cnt = 0, c_prevnw = 0;                           // letters (mod 4) of the run ending at pos0-1; nonWS[pos0-1]
  if (pos0 > 0) {
    c_prevnw = !is_ws_scalar(bytes[pos0 - 1]);
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
  long long last_o = -1;              // largest boundary seen (validation of monotonicity across windows)

  // boundary window: lane holds off[kb + lane]
  long long o = kInfOff;
  auto load_window = [&]() {
    const long long idx = kb + lane;
    o = idx < nb_total ? off[idx] : kInfOff;
    long long prev = __shfl_up_sync(kFull, o, 1);
    if (lane == 0) prev = last_o;
    if (idx < nb_total && (o < 0 || o > n_bytes || o < prev)) atomicOr(status, DS_DEV_BAD_OFFSETS);
  };
  load_window();

  const int rot = (lane >> 1) & 3;    // 16-byte pieces are read in rotated order: conflict-free LDS.128 at a 64-byte lane stride
  static_assert((kStages & (kStages - 1)) == 0, "kStages must be a power of two");
  long long cs = pos0;
  for (unsigned it = 0; it < n_it; ++it, cs += kChunk) {
    const int s = (int)(it & (kStages - 1));
    const unsigned parity = (it / kStages) & 1u;
    const long long ce = cs + kChunk;   // chunk = positions [cs,ce) relative to bytes

    // (a) prompt boundaries inside this chunk -> start bits (lanes 0..nb-1 of the window hold them)
    bool inb = o >= cs && o < ce;
    unsigned bm = __ballot_sync(kFull, inb);
    if (inb) atomicOr(&sb[(int)(o - cs) >> 5], 1u << ((int)(o - cs) & 31));
    if (bm == kFull) {                                   // rare: more than 32 boundaries may fall into one chunk
      for (long long kk = kb + 32; kk < nb_total; kk += 32) {
        const long long idx = kk + lane;
        const long long o2 = idx < nb_total ? off[idx] : kInfOff;
        const bool in2 = o2 >= cs && o2 < ce;
        if (in2) atomicOr(&sb[(int)(o2 - cs) >> 5], 1u << ((int)(o2 - cs) & 31));
        if (__ballot_sync(kFull, in2) != kFull) break;
      }
    }

    // (b) wait for the chunk, classify own 64 bytes
    mbar_wait(&mbar[s], parity);
    const uint8_t* seg = stage[s] + lane * kSeg;
    uint32_t wf[4], df[4];                               // 128 x (16-bit mask) of piece (j+rot)&3
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int r = (j + rot) & 3;
      const uint4 v = *reinterpret_cast<const uint4*>(seg + r * 16);
      uint32_t w0, w1, w2, w3, e0, e1, e2, e3;
      classify4(v.x, one, w0, e0); classify4(v.y, one, w1, e1); classify4(v.z, one, w2, e2); classify4(v.w, one, w3, e3);
      wf[j] = mask8x128(w2, w3) * 256u + mask8x128(w0, w1);
      df[j] = mask8x128(e2, e3) * 256u + mask8x128(e0, e1);
    }
    __syncwarp();
    if (lane == 0 && it + kStages < n_it) issue(it + kStages);   // the stage's bytes are all in registers now
    unsigned long long ws = rotl16(wf[1] * 512u + (wf[0] >> 7), wf[3] * 512u + (wf[2] >> 7), rot);
    unsigned long long d = rotl16(df[1] * 512u + (df[0] >> 7), df[3] * 512u + (df[2] >> 7), rot);
    if (cs < 0 || ce > n_bytes) {                        // bytes outside [0,n_bytes) count as whitespace
      const long long sp = cs + (long long)lane * kSeg;
      long long lo = -sp, hi = n_bytes - sp;
      lo = lo < 0 ? 0 : (lo > 64 ? 64 : lo);
      hi = hi < 0 ? 0 : (hi > 64 ? 64 : hi);
      unsigned long long valid = 0ull;
      if (hi > lo) valid = (hi == 64 ? ~0ull : ((1ull << hi) - 1ull)) & ~((1ull << lo) - 1ull);
      ws |= ~valid; d |= ~valid;
    }
    const unsigned long long S = *reinterpret_cast<const unsigned long long*>(sb + 2 * lane);
    *reinterpret_cast<unsigned long long*>(sb + 2 * lane) = 0ull;

    // (c) letter-run summary of this segment and the carries between lanes
    const unsigned long long L = ~d, nonws = ~ws;
    const unsigned long long cont = L & ~S & ((L << 1) | 1ull);   // letter that continues the previous byte's run
    const bool has_break = cont != ~0ull;
    unsigned cnt_out = 0;
    if (has_break) {
      const int k = clz64(~cont);                                 // trailing continuation bytes
      cnt_out = (unsigned)(k + (int)((L >> (63 - k)) & 1ull)) & 3u;
    }
    const unsigned brk_mask = __ballot_sync(kFull, has_break);
    const unsigned below = brk_mask & ((1u << lane) - 1u);
    const unsigned from_lane = __shfl_sync(kFull, cnt_out, below ? 31 - __clz(below) : 0);
    const unsigned cnt_in = below ? from_lane : c_cnt;
    unsigned prevnw = __shfl_up_sync(kFull, (unsigned)(nonws >> 63), 1);
    if (lane == 0) prevnw = c_prevnw;
    c_prevnw = __shfl_sync(kFull, (unsigned)(nonws >> 63), 31);
    if (brk_mask) c_cnt = __shfl_sync(kFull, cnt_out, 31 - __clz(brk_mask));   // else unchanged: 2048 = 0 (mod 4)

    // (d) flags
    const unsigned long long fwm = nonws & (S | ~((nonws << 1) | (unsigned long long)prevnw));
    unsigned long long F = L & ~cont;                             // run starts
    if (cont & 1ull) {                                            // the carried-in run's next multiple-of-4 position
      const unsigned q = (4u - cnt_in) & 3u;
      const unsigned long long mq = (2ull << q) - 1ull;
      if ((cont & mq) == mq) F |= 1ull << q;
    }
    unsigned long long P = cont & (cont << 1) & (cont << 2) & (cont << 3);
    F |= (F << 4) & P;  P &= P << 4;
    F |= (F << 8) & P;  P &= P << 8;
    F |= (F << 16) & P; P &= P << 16;
    F |= (F << 32) & P;
    const unsigned long long ftm = F | (d & ~ws);
    const unsigned own = (unsigned)__popcll(fwm) | ((unsigned)__popcll(ftm) << 16);
    const unsigned total = __reduce_add_sync(kFull, own);         // <= 2048 per field: no carry between the halves

    // (e) attribute to prompts: boundary k (= off[k]) closes prompt k-1
    unsigned base_c = 0;                                          // packed prefix count at the last boundary handled
    if (bm) {
      unsigned incl = own;                                        // inclusive prefix over lanes
#pragma unroll
      for (int sft = 1; sft < 32; sft <<= 1) {
        const unsigned y = __shfl_up_sync(kFull, incl, sft);
        if (lane >= sft) incl += y;
      }
      const unsigned cum = incl - own;
      for (;;) {
        const int nb = __popc(bm);
        const int rel = inb ? (int)(o - cs) : 0;
        const int t = rel >> 6, bit = rel & 63;
        const unsigned cum_t = __shfl_sync(kFull, cum, t);
        const unsigned long long fw_t = shfl64(fwm, t), ft_t = shfl64(ftm, t);
        const unsigned long long mk = (1ull << bit) - 1ull;
        const unsigned cj = cum_t + (unsigned)__popcll(fw_t & mk) + ((unsigned)__popcll(ft_t & mk) << 16);
        unsigned prev = __shfl_up_sync(kFull, cj, 1);
        if (lane == 0) prev = base_c;
        const unsigned dlt = cj - prev;                           // both fields are non-decreasing: no borrow
        unsigned nwd = dlt & 0xffffu, ntk = dlt >> 16;
        const long long p = kb + lane - 1;                        // prompt closed by this lane's boundary
        if (lane == 0) { nwd += accW; ntk += accT; }
        if (inb && p >= 0) {
          if (lane == 0 && open_before_span) {
            if (nwd) atomicAdd(words + p, (int)nwd);
            if (ntk) atomicAdd(tokens + p, (int)ntk);
          } else {
            words[p] = (int)nwd; tokens[p] = (int)ntk;
          }
        }
        accW = 0; accT = 0; open_before_span = false;
        base_c = __shfl_sync(kFull, cj, nb - 1);
        last_o = __shfl_sync(kFull, o, nb - 1);
        kb += nb;
        load_window();
        if (nb < 32) break;
        inb = o >= cs && o < ce;
        bm = __ballot_sync(kFull, inb);
        if (!bm) break;
      }
    }
    const unsigned tail = total - base_c;
    accW += tail & 0xffffu; accT += tail >> 16;
    __syncwarp();
  }

  // the prompt still open at the span's end continues in the next warp's span
  if (lane == 0 && kb >= 1 && kb <= n_prompts) {
    if (accW) atomicAdd(words + (kb - 1), (int)accW);
    if (accT) atomicAdd(tokens + (kb - 1), (int)accT);
  }
}

}  // namespace k1

size_t ws_characterize(int64_t, int64_t) { return 256; }

}  // namespace ds

extern "C" int ds_characterize(const uint8_t* bytes, int64_t n_bytes, const int64_t* offsets, int64_t n_prompts,
                               int32_t* words_out, int32_t* tokens_out, void* workspace, size_t workspace_bytes, void* stream) {
  using namespace ds;
  (void)workspace; (void)workspace_bytes;
  if (n_bytes < 0 || n_prompts < 0) return DS_EINVAL;
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
  const long long n_chunks = (mis + n_bytes + k1::kChunk - 1) / k1::kChunk;
  static bool attr_set = false;
  if (!attr_set) {
    DS_CUDA(cudaFuncSetAttribute(k1::characterize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(k1::Smem)));
    attr_set = true;
  }
  long long grid = (long long)kNumSMs * k1::kCtasPerSM;
  const long long need = (n_chunks + k1::kWarps - 1) / k1::kWarps;
  if (grid > need) grid = need;
  k1::characterize_kernel<<<(unsigned)grid, k1::kThreads, sizeof(k1::Smem), st>>>(bytes, n_bytes, offsets, n_prompts, words_out,
                                                                               tokens_out, n_chunks, status, 1u);
  note_launch();
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}
