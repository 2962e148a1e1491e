// K1 — ds_characterize: single-pass HBM stream over packed prompt text (SURVEY.md §8(a) a1+a2).
//
// Definition (include/driftsched.h):
//   words[i]  = # maximal runs of non-WS bytes in prompt i
//   tokens[i] = # PUNCT bytes + sum over maximal LETTER runs of ceil(len/4)
// Per-byte flag form used here (equivalent, proven in DESIGN.md §6.1):
//   wordstart[j] = nonWS[j] && (j starts a prompt || WS[j-1])
//   tokflag[j]   = PUNCT[j] || (LETTER[j] && (# letters before j in its run, runs reset at prompt starts) % 4 == 0)
//   words[i] = popcount(wordstart over [a,b)),  tokens[i] = popcount(tokflag over [a,b)).
//
// Design (B200): persistent CTAs, each owning one contiguous span of 16 KiB tiles; tiles are brought into shared
// memory by 1-D TMA bulk copies (cp.async.bulk + mbarrier, kStages deep) so the LSU pipe carries no global loads;
// every thread owns 64 contiguous bytes, classifies them 4 at a time with SWAR threshold adds (11 adds + 6 LOP3
// per word), compacts the per-byte class bits to 64-bit masks (PRMT + IDP4A), derives both flag masks with
// bit-parallel logic (Kogge-Stone stride-4 propagation for the mod-4 run position) and a 2-bit carry that
// composes across lanes / warps / tiles; prompts are attributed through a per-tile prefix of popcounts, plain
// stores for prompts inside a tile and integer atomicAdd only for prompts that straddle a tile edge.
#include "common.cuh"

namespace ds {
namespace k1 {

constexpr int kThreads = 256;
constexpr int kSeg = 64;                      // bytes per thread
constexpr int kTile = kThreads * kSeg;        // 16 KiB
constexpr int kStages = 4;
constexpr int kWarps = kThreads / 32;
constexpr int kCtasPerSM = 2;

struct Smem {
  alignas(128) uint8_t data[kStages][kTile];
  unsigned long long mbar[kStages];
  unsigned long long sbits[kThreads];   // prompt-start bit per byte of the current tile
  unsigned long long fw[kThreads];      // word-start flags
  unsigned long long ft[kThreads];      // token flags
  unsigned int cum[kThreads];           // exclusive in-warp prefix of (popc(fw) | popc(ft)<<16)
  unsigned int wtot[kWarps];            // per-warp totals (packed)
  unsigned int wsum[kWarps];            // per-warp letter-run summary: bit2 = has break, bits0-1 = tail count mod 4
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
// (z - n*0x01010101) is (low7(x) >= n). Intervals are XORs of nested thresholds. Bytes >= 0x80 are LETTER (& ~x).
__device__ __forceinline__ void classify4(uint32_t x, uint32_t& ws7, uint32_t& d7) {
  const uint32_t z = x | 0x80808080u;
  const uint32_t t9 = z - 0x09090909u, t14 = z - 0x0E0E0E0Eu, t32 = z - 0x20202020u, t33 = z - 0x21212121u;
  const uint32_t t48 = z - 0x30303030u, t58 = z - 0x3A3A3A3Au, t65 = z - 0x41414141u, t91 = z - 0x5B5B5B5Bu;
  const uint32_t t97 = z - 0x61616161u, t123 = z - 0x7B7B7B7Bu, t127 = z - 0x7F7F7F7Fu;
  const uint32_t s1 = t9 ^ t14 ^ t32;                       // [9,13] u [32,..)
  ws7 = (s1 ^ t33) & ~x;                                    // WS = [9,13] u {32}
  d7 = (s1 ^ (t48 ^ t58 ^ t65) ^ (t91 ^ t97 ^ t123) ^ t127) & ~x;  // non-LETTER = WS u PUNCT
}

// bit 7 of each byte of (w0,w1) -> 8-bit mask, returned NEGATED (IDP4A with signed 0xFF bytes)
__device__ __forceinline__ int movemask8_neg(uint32_t w0, uint32_t w1) {
  uint32_t c0, c1;   // selector nibble 8+i replicates the sign bit of byte i (__byte_perm drops that bit, prmt.b32 keeps it)
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(c0) : "r"(w0), "r"(0u), "r"(0xba98u));
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(c1) : "r"(w1), "r"(0u), "r"(0xba98u));
  int acc;
  asm("dp4a.s32.u32 %0, %1, %2, %3;" : "=r"(acc) : "r"(c0), "r"(0x08040201u), "r"(0));
  asm("dp4a.s32.u32 %0, %1, %2, %3;" : "=r"(acc) : "r"(c1), "r"(0x80402010u), "r"(acc));
  return acc;
}

__device__ __forceinline__ bool is_ws_scalar(uint32_t c) { return (c - 9u) <= 4u || c == 32u; }
__device__ __forceinline__ bool is_letter_scalar(uint32_t c) {
  bool punct = (c - 0x21u) <= 0x0Eu || (c - 0x3Au) <= 6u || (c - 0x5Bu) <= 5u || (c - 0x7Bu) <= 3u;
  return !punct && !is_ws_scalar(c);
}


#ifdef DS_DEBUG
__device__ unsigned long long ds_dbg[256 * 8];
#endif
__device__ __forceinline__ int clz64(unsigned long long v) { return __clzll((long long)v); }

// max k in [0,n) with off[k] <= pos (0 if none); executed by one full warp, 32-ary search
__device__ __forceinline__ long long warp_search_le(const int64_t* __restrict__ off, long long n, long long pos, int lane) {
  long long lo = 0, hi = n;  // answer in [lo,hi) if any
  if (n <= 0) return 0;
  while (hi - lo > 1) {
    long long stride = (hi - lo + 31) / 32;
    long long k = lo + (long long)lane * stride;
    bool pred = (k < hi) && (off[k] <= pos);
    unsigned m = __ballot_sync(0xffffffffu, pred);
    int c = __popc(m);  // predicates form a prefix (offsets non-decreasing)
    if (c == 0) return 0;
    long long nlo = lo + (long long)(c - 1) * stride;
    long long nhi = lo + (long long)c * stride;
    lo = nlo;
    hi = nhi < hi ? nhi : hi;
  }
  return lo;
}

__global__ void __launch_bounds__(kThreads, kCtasPerSM)
characterize_kernel(const uint8_t* __restrict__ bytes, long long n_bytes, const int64_t* __restrict__ off, long long n_prompts,
                    int32_t* __restrict__ words, int32_t* __restrict__ tokens, long long n_tiles, unsigned int* status) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  Smem& sm = *reinterpret_cast<Smem*>(smem_raw);
  __shared__ long long sh_pfirst;
  __shared__ unsigned int sh_cnt[2], sh_prevnw[2];

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const unsigned long long base = (unsigned long long)bytes;
  const long long mis = (long long)(base & 15ull);
  const uint8_t* abase = bytes - mis;                         // 16-byte aligned
  const long long load_end = (mis + n_bytes + 15) & ~15ll;    // bytes from abase that may be read
  const long long t_begin = (long long)blockIdx.x * n_tiles / gridDim.x;
  const long long t_end = (long long)(blockIdx.x + 1) * n_tiles / gridDim.x;
  if (t_begin >= t_end) return;

  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&sm.mbar[s], 1);
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  }
  sm.sbits[tid] = 0ull;
  __syncthreads();

  auto issue = [&](long long t) {  // thread 0 only
    const int s = (int)((t - t_begin) % kStages);
    long long a0 = t * (long long)kTile;
    long long len = load_end - a0;
    if (len > kTile) len = kTile;
    mbar_expect_tx(&sm.mbar[s], (unsigned)len);
    tma_load_1d(sm.data[s], abase + a0, (unsigned)len, &sm.mbar[s]);
  };
  if (tid == 0)
    for (long long t = t_begin; t < t_end && t < t_begin + kStages - 1; ++t) issue(t);

  // span prologue: first overlapping prompt, and the carries at the span's first byte
  const long long pos0 = t_begin * (long long)kTile - mis;
  if (warp == 0) {
    long long pf = warp_search_le(off, n_prompts, pos0, lane);
    unsigned cnt = 0, pnw = 0;
    if (pos0 > 0) {
      pnw = !is_ws_scalar(bytes[pos0 - 1]);
      long long lb = off[pf];                 // letters before pos0 count only back to the prompt's start
      if (lb < 0) lb = 0;
      long long k = pos0 - 1;
      bool found = false;
      while (!found && k >= lb) {
        long long j = k - lane;
        bool brk = (j < lb) || !is_letter_scalar(bytes[j]);
        unsigned m = __ballot_sync(0xffffffffu, brk);
        if (m) { cnt += __ffs(m) - 1; found = true; } else { cnt += 32; k -= 32; }
      }
      cnt &= 3u;
    }
    if (lane == 0) { sh_pfirst = pf; sh_cnt[0] = cnt; sh_prevnw[0] = pnw; }
  }
  __syncthreads();
  long long p_first = sh_pfirst;

  for (long long t = t_begin; t < t_end; ++t) {
    const long long it = t - t_begin;
    const int s = (int)(it % kStages);
    const unsigned parity = (unsigned)((it / kStages) & 1);
    const int par = (int)(it & 1);
    const long long ts = t * (long long)kTile - mis, te = ts + kTile;
    if (tid == 0 && t + kStages - 1 < t_end) issue(t + kStages - 1);

    // (a) prefetch this thread's first candidate offset
    long long p_mine = p_first + tid;
    long long o_pref = (p_mine < n_prompts) ? off[p_mine] : 0;

    // (b,c) wait for the tile, classify own 64 bytes. chunk order rotated by lane>>1: conflict-free LDS.128
    mbar_wait(&sm.mbar[s], parity);
    const uint8_t* seg = sm.data[s] + tid * kSeg;
    uint32_t ws_lo = 0, ws_hi = 0, d_lo = 0, d_hi = 0;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int r = (j + (lane >> 1)) & 3;
      const uint4 v = *reinterpret_cast<const uint4*>(seg + r * 16);
      uint32_t w0, w1, w2, w3, e0, e1, e2, e3;
      classify4(v.x, w0, e0); classify4(v.y, w1, e1); classify4(v.z, w2, e2); classify4(v.w, w3, e3);
      const int wa = movemask8_neg(w0, w1), wb = movemask8_neg(w2, w3);
      const int da = movemask8_neg(e0, e1), db = movemask8_neg(e2, e3);
      const uint32_t wm = (uint32_t)(-(wa + (wb << 8))), dm = (uint32_t)(-(da + (db << 8)));  // 16-bit masks
      const uint32_t sh = (r & 1) * 16;
      if (r & 2) { ws_hi |= wm << sh; d_hi |= dm << sh; } else { ws_lo |= wm << sh; d_lo |= dm << sh; }
    }
    unsigned long long ws = ((unsigned long long)ws_hi << 32) | ws_lo, d = ((unsigned long long)d_hi << 32) | d_lo;
    {  // bytes outside [0,n_bytes) count as whitespace
      const long long sp = ts + (long long)tid * kSeg;
      if (sp < 0 || sp + kSeg > n_bytes) {
        unsigned long long valid = 0ull;
        for (int j = 0; j < kSeg; ++j) if (sp + j >= 0 && sp + j < n_bytes) valid |= 1ull << j;
        ws |= ~valid; d |= ~valid;
      }
    }

    // (d) pass A: prompt-start bits of this tile, and how many prompts begin at or before the tile's end
    long long n_le = 0;
    for (int chunk = 0;; ++chunk) {
      const long long p = p_first + (long long)chunk * kThreads + tid;
      const bool in = p < n_prompts;
      const long long o = chunk == 0 ? o_pref : (in ? off[p] : 0);
      if (in && o >= ts && o < te) atomicOr(&sm.sbits[(o - ts) >> 6], 1ull << ((o - ts) & 63));
      const int c = __syncthreads_count(in && o <= te);
      n_le += c;
      if (c < kThreads) break;
    }

    // (e) letter-run summary of this segment
    const unsigned long long S = sm.sbits[tid];
    sm.sbits[tid] = 0ull;
    const unsigned long long L = ~d, nonws = ~ws;
    const unsigned long long cont = L & ~S & ((L << 1) | 1ull);   // letter that continues the previous byte's run
    const bool has_break = cont != ~0ull;
    unsigned cnt_out = 0;
    if (has_break) {
      const int k = clz64(~cont);                                 // trailing continuation bytes
      cnt_out = (unsigned)(k + (int)((L >> (63 - k)) & 1ull)) & 3u;
    }
    const unsigned brk_mask = __ballot_sync(0xffffffffu, has_break);
    const int last_brk = brk_mask ? 31 - __clz(brk_mask) : 0;
    const unsigned warp_tail = __shfl_sync(0xffffffffu, cnt_out, last_brk);
    if (lane == 0) sm.wsum[warp] = (brk_mask ? 4u : 0u) | warp_tail;
    if (tid == kThreads - 1) sh_prevnw[par ^ 1] = (unsigned)(nonws >> 63);
    __syncthreads();  // sync2

    // (g) carries
    unsigned warp_in = sh_cnt[par];
    {
      bool got = false;
      for (int w = warp - 1; w >= 0 && !got; --w) {
        const unsigned u = sm.wsum[w];
        if (u & 4u) { warp_in = u & 3u; got = true; }
      }
    }
    if (tid == kThreads - 1) sh_cnt[par ^ 1] = brk_mask ? warp_tail : warp_in;
    const unsigned below = brk_mask & ((1u << lane) - 1u);
    const unsigned from_lane = __shfl_sync(0xffffffffu, cnt_out, below ? 31 - __clz(below) : 0);
    const unsigned cnt_in = below ? from_lane : warp_in;

    unsigned prevnw = __shfl_up_sync(0xffffffffu, (unsigned)(nonws >> 63), 1);
    if (lane == 0) {
      if (tid == 0) prevnw = sh_prevnw[par];
      else {
        const long long pp = ts + (long long)tid * kSeg - 1;
        prevnw = (pp >= 0 && pp < n_bytes) ? !is_ws_scalar(seg[-1]) : 0u;
      }
    }

    // word starts
    const unsigned long long fwm = nonws & (S | ~((nonws << 1) | (unsigned long long)prevnw));
    // token flags: run starts, the carried-in run's next 4-boundary, then stride-4 propagation along each run
    unsigned long long F = L & ~cont;
    if (cont & 1ull) {
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

    // (g2) per-tile prefix of popcounts
    const unsigned own = (unsigned)__popcll(fwm) | ((unsigned)__popcll(ftm) << 16);
    unsigned incl = own;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned y = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += y;
    }
#ifdef DS_DEBUG
    if (blockIdx.x == 0 && t == t_begin) { ds_dbg[tid * 8 + 0] = ws; ds_dbg[tid * 8 + 1] = d; ds_dbg[tid * 8 + 2] = S; ds_dbg[tid * 8 + 3] = fwm;
      ds_dbg[tid * 8 + 4] = ftm; ds_dbg[tid * 8 + 5] = cnt_in; ds_dbg[tid * 8 + 6] = *reinterpret_cast<const unsigned long long*>(seg); ds_dbg[tid * 8 + 7] = n_le; }
#endif
    sm.fw[tid] = fwm; sm.ft[tid] = ftm; sm.cum[tid] = incl - own;
    if (lane == 31) sm.wtot[warp] = incl;
    __syncthreads();  // sync3

    // (i) pass B: attribute to prompts
    for (long long q = tid; q < n_le; q += kThreads) {
      const long long p = p_first + q;
      const long long a = off[p], b = off[p + 1];
      if (b < a || a < 0 || b > n_bytes) { atomicOr(status, DS_DEV_BAD_OFFSETS); continue; }
      const long long lo = a > ts ? a : ts, hi = b < te ? b : te;
      if (lo >= hi) continue;
      unsigned c[2];
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int x = (int)((e ? hi : lo) - ts);      // 0..kTile
        int sg = x >> 6, nb = x & 63;
        if (sg == kThreads) { sg = kThreads - 1; nb = 64; }
        const unsigned long long mk = nb == 64 ? ~0ull : ((1ull << nb) - 1ull);
        unsigned v = sm.cum[sg] + (unsigned)__popcll(sm.fw[sg] & mk) + ((unsigned)__popcll(sm.ft[sg] & mk) << 16);
        for (int w = 0; w < (sg >> 5); ++w) v += sm.wtot[w];
        c[e] = v;
      }
      const unsigned dlt = c[1] - c[0];
      const int nw = (int)(dlt & 0xffffu), nt = (int)(dlt >> 16);
      if (a >= ts && b <= te) { words[p] = nw; tokens[p] = nt; }
      else { if (nw) atomicAdd(words + p, nw); if (nt) atomicAdd(tokens + p, nt); }
    }
    if (n_le > 0) p_first += n_le - 1;
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
  const long long n_tiles = (mis + n_bytes + k1::kTile - 1) / k1::kTile;
  static bool attr_set = false;
  if (!attr_set) {
    DS_CUDA(cudaFuncSetAttribute(k1::characterize_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(k1::Smem)));
    attr_set = true;
  }
  long long grid = (long long)kNumSMs * k1::kCtasPerSM;
  if (grid > n_tiles) grid = n_tiles;
  k1::characterize_kernel<<<(unsigned)grid, k1::kThreads, sizeof(k1::Smem), st>>>(bytes, n_bytes, offsets, n_prompts, words_out,
                                                                               tokens_out, n_tiles, status);
  note_launch();
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}
