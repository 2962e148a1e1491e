// K3 — ds_latencies + ds_tail_stats (Tables VI-VIII).
//
// ds_tail_stats: segmented nearest-rank percentiles by MSB-first radix select on 8-bit digits. Keys are the
// values with the sign bit flipped (unsigned order == signed order). Pass 0 counts each segment and reduces
// AND / OR of all keys: a digit on which every key agrees is skipped (latencies < 2^40 ticks skip 3 of 8).
// Per digit: histogram kernel (shared-memory privatised when (segments x percentiles x 256) fits, global
// atomics otherwise) -> select kernel (one thread per (segment, percentile) walks 256 bins, fixes the digit,
// reduces the rank). Traffic: 12 B per value per non-skipped digit; only keys matching the prefix are counted.
#include "common.cuh"
#include <mutex>
#include <type_traits>

namespace ds {
namespace k3 {

#ifndef DS_K3_KEYS
#define DS_K3_KEYS 16    // staged keys per thread and trip of the digit passes: 4 / 8 / 16 = configs[3] stats at 4096 traces 16.05 / 13.94 / 13.57 ms
#endif
static_assert(DS_K3_KEYS % 4 == 0, "16-byte key loads");

constexpr int kMaxPct = 8;
constexpr unsigned long long kSign = 0x8000000000000000ull;

struct Ws {               // header at the start of the workspace
  unsigned long long and_bits, or_bits;
  unsigned int any;
  unsigned int nostage;   // ds_latency_stats: the staged keys are unusable (no room, or out_off is not a partition)
};
// Digits are aligned to the highest bit on which the keys differ (diff = AND ^ OR of all keys): pass j = 0, 1, ... covers
// bits [top - 8(j+1), top - 8j) clamped at 0, top = number of low bits that vary. A fixed alignment (bits 56-63, 48-55, ...)
// wastes a full-cost pass on a top digit that carries one or two bits (25-bit latencies: bits 24-31 hold one bit).
struct DigitPos { int lo, width; bool active; };
__device__ __forceinline__ int vary_top(unsigned long long diff) { return diff ? 64 - __clzll((long long)diff) : 0; }
__device__ __forceinline__ DigitPos digit_pos(unsigned long long diff, int j) {
  DigitPos p;
  const int hi_end = vary_top(diff) - 8 * j;
  p.active = hi_end > 0;
  p.lo = hi_end > 8 ? hi_end - 8 : 0;
  p.width = p.active ? hi_end - p.lo : 0;
  return p;
}
// layout: Ws | counts[n_seg] u64 | prefix[n_seg*n_pct] u64 | rank[n_seg*n_pct] u64 | hist[n_seg*n_pct*256] u32
struct Layout {
  Ws* hdr; unsigned long long* counts; unsigned long long* prefix; unsigned long long* rank; unsigned int* hist;
  size_t total;
};
inline Layout make_layout(void* base, int64_t n_seg, int64_t n_pct) {
  Layout L; char* p = (char*)base; size_t o = 0;
  L.hdr = (Ws*)(p + o); o += 256;
  L.counts = (unsigned long long*)(p + o); o += align_up(8 * (size_t)n_seg, 256);
  L.prefix = (unsigned long long*)(p + o); o += align_up(8 * (size_t)(n_seg * n_pct), 256);
  L.rank = (unsigned long long*)(p + o); o += align_up(8 * (size_t)(n_seg * n_pct), 256);
  L.hist = (unsigned int*)(p + o); o += align_up(4 * 256 * (size_t)(n_seg * n_pct), 256);
  L.total = o;
  return L;
}

__global__ void latencies_kernel(const int64_t* __restrict__ trace_off, const int64_t* __restrict__ arrival,
                                 const uint8_t* __restrict__ tier, const ds_instance* __restrict__ inst,
                                 const int64_t* __restrict__ out_off, const int64_t* __restrict__ arr_ov,
                                 const int64_t* __restrict__ start,
                                 const int64_t* __restrict__ done, const int32_t* __restrict__ group,
                                 const int64_t* __restrict__ t_mid, int64_t* __restrict__ e2e, int64_t* __restrict__ qd,
                                 int32_t* __restrict__ seg_tier, int32_t* __restrict__ seg_all) {
  const long long ii = blockIdx.x;
  const int t = inst[ii].trace;
  const long long lo = trace_off[t], n = trace_off[t + 1] - lo, oo = out_off[ii];
  const int g0 = group ? group[ii] : 0;
  const bool ph = t_mid != nullptr;
  const long long tm = ph ? t_mid[t] : 0;
  const int64_t* __restrict__ ap = arr_ov ? arr_ov + oo : arrival + lo;   // closed loop: the instance's own arrival ticks
  for (long long r = threadIdx.x; r < n; r += blockDim.x) {
    const long long a = ap[r];
    e2e[oo + r] = done[oo + r] - a;
    qd[oo + r] = start[oo + r] - a;
    const int g = ph ? g0 * 2 + (a >= tm ? 1 : 0) : g0;
    if (seg_tier) seg_tier[oo + r] = g * 3 + tier[lo + r];
    if (seg_all) seg_all[oo + r] = g;
  }
}

// Histogram add in shared memory: a plain atomic by every lane whose predicate holds. Round 1 aggregated the lanes of a warp
// first (leader's bin by broadcast + ballot, one atomic for all lanes that hit it), on the assumption that keys sharing
// their high digits serialise 32-way on one bin. Measured again in r02 on B200 (20 M keys per call): spread keys 0.65 ->
// 0.57 ms, keys that are all equal but 0.5 % outliers 1.33 -> 0.70 ms, two distinct values 1.32 -> 0.72 ms, and the stats
// stage of configs[3] -35 %: same-address shared-memory atomics of a warp are combined by the hardware, and the two ballots
// and the shuffle per add were what the passes spent their issue slots on.
__device__ __forceinline__ void hist_add(unsigned int* bins, bool pred, unsigned bin) {
  if (pred) atomicAdd(&bins[bin], 1u);
}

constexpr int kMaxSegPct = 200;   // (segments x percentiles) of the fused pass: 200 KB of shared-memory histograms at most
constexpr int kUnroll = 4;   // independent 12-byte loads in flight per thread

__global__ void __launch_bounds__(512) count_kernel(const int64_t* __restrict__ v, const int32_t* __restrict__ seg, long long n, int n_seg,
                             Ws* hdr, unsigned long long* counts) {
  extern __shared__ unsigned int sc[];   // per-block segment counts when n_seg is small
  const bool priv = n_seg <= 4096;
  if (priv) { for (int i = threadIdx.x; i < n_seg; i += blockDim.x) sc[i] = 0; __syncthreads(); }
  unsigned long long a = ~0ull, o = 0ull; bool any = false;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long base = blockIdx.x * (long long)blockDim.x; base < n; base += stride * kUnroll) {   // block-uniform trip count
    int sv[kUnroll]; unsigned long long kv[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const long long i = base + u * stride + threadIdx.x;
      sv[u] = i < n ? seg[i] : -1;
      kv[u] = i < n ? (unsigned long long)v[i] ^ kSign : 0ull;
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const bool ok = sv[u] >= 0 && sv[u] < n_seg;
      if (ok) { a &= kv[u]; o |= kv[u]; any = true; }
      if (priv) hist_add(sc, ok, (unsigned)sv[u]);
      else if (ok) atomicAdd(&counts[sv[u]], 1ull);
    }
  }
  for (int d = 16; d > 0; d >>= 1) { a &= __shfl_xor_sync(0xffffffffu, a, d); o |= __shfl_xor_sync(0xffffffffu, o, d); }
  const unsigned anym = __ballot_sync(0xffffffffu, any);
  if ((threadIdx.x & 31) == 0 && anym) { atomicAnd(&hdr->and_bits, a); atomicOr(&hdr->or_bits, o); atomicOr(&hdr->any, 1u); }
  if (priv) { __syncthreads(); for (int i = threadIdx.x; i < n_seg; i += blockDim.x) if (sc[i]) atomicAdd(&counts[i], (unsigned long long)sc[i]); }
}

struct Pcts { int p[kMaxPct]; };

__global__ void init_kernel(const unsigned long long* counts, int n_seg, int n_pct, Pcts pc, const Ws* hdr, unsigned long long* prefix,
                            unsigned long long* rank, int64_t* count_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n_seg * n_pct) return;
  const int s = i / n_pct, q = i % n_pct;
  const unsigned long long c = counts[s];
  unsigned long long r = ((unsigned long long)pc.p[q] * c + 99ull) / 100ull;   // nearest rank (A13)
  if (r < 1) r = 1;
  if (r > c) r = c;
  const int top = vary_top(hdr->and_bits ^ hdr->or_bits);           // the bits above `top` are common to all keys
  prefix[i] = (hdr->any && top < 64) ? hdr->and_bits >> top : 0ull; rank[i] = r;
  if (q == 0 && count_out) count_out[s] = (int64_t)c;
}

// digit d (7 = most significant). Keys whose bits above digit d equal prefix[s,q] are counted in hist[s,q][digit].
template <bool kPriv>
__global__ void __launch_bounds__(512) hist_kernel(const int64_t* __restrict__ v, const int32_t* __restrict__ seg, long long n, int n_seg,
                            int n_pct, int d, const Ws* hdr, const unsigned long long* __restrict__ prefix, unsigned int* hist) {
  const DigitPos dp = digit_pos(hdr->and_bits ^ hdr->or_bits, 7 - d);
  if (!hdr->any || !dp.active) return;                           // no varying bits left for this pass
  extern __shared__ unsigned int sh[];
  const int nb = n_seg * n_pct * 256;
  if (kPriv) { for (int i = threadIdx.x; i < nb; i += blockDim.x) sh[i] = 0; __syncthreads(); }
  unsigned int* bins = kPriv ? sh : hist;
  const int shift = dp.lo, hshift = dp.lo + dp.width;
  const unsigned dmask = (1u << dp.width) - 1u;
  const long long stride = (long long)gridDim.x * blockDim.x;
  for (long long base = blockIdx.x * (long long)blockDim.x; base < n; base += stride * kUnroll) {   // block-uniform trip count
    int sv[kUnroll]; unsigned long long kv[kUnroll];
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const long long i = base + u * stride + threadIdx.x;
      sv[u] = i < n ? seg[i] : -1;
      kv[u] = i < n ? (unsigned long long)v[i] ^ kSign : 0ull;
    }
#pragma unroll
    for (int u = 0; u < kUnroll; ++u) {
      const bool ok = sv[u] >= 0 && sv[u] < n_seg;
      const int s = ok ? sv[u] : 0;
      const unsigned long long hi = hshift >= 64 ? 0ull : (kv[u] >> hshift);
      const unsigned dig = (unsigned)(kv[u] >> shift) & dmask;
      for (int q = 0; q < n_pct; ++q)
        hist_add(bins, ok && hi == prefix[s * n_pct + q], (unsigned)((s * n_pct + q) * 256) + dig);
    }
  }
  if (kPriv) { __syncthreads(); for (int i = threadIdx.x; i < nb; i += blockDim.x) if (sh[i]) atomicAdd(&hist[i], sh[i]); }
}

// one warp per (segment, percentile): lane l owns bins 8l..8l+7; warp prefix scan finds the digit that holds the rank
__global__ void select_kernel(int n_seg, int n_pct, int d, const Ws* hdr, const unsigned long long* counts,
                              unsigned long long* prefix, unsigned long long* rank, unsigned int* hist, int64_t* out) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5, lane = threadIdx.x & 31;
  if (i >= n_seg * n_pct) return;
  const DigitPos dp = digit_pos(hdr->and_bits ^ hdr->or_bits, 7 - d);
  const bool skip = !hdr->any || !dp.active;
  unsigned long long pf = prefix[i];
  if (!skip) {
    uint4* h4 = reinterpret_cast<uint4*>(hist + (size_t)i * 256 + lane * 8);
    const uint4 x = h4[0], y = h4[1];
    h4[0] = make_uint4(0, 0, 0, 0); h4[1] = make_uint4(0, 0, 0, 0);   // ready for the next digit
    const unsigned c[8] = {x.x, x.y, x.z, x.w, y.x, y.y, y.z, y.w};
    unsigned long long own = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) own += c[k];
    unsigned long long incl = own;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned long long t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    const unsigned long long r = rank[i];
    const unsigned hit = __ballot_sync(0xffffffffu, incl >= r);   // first lane whose inclusive count reaches the rank
    const int src = hit ? __ffs(hit) - 1 : 31;
    unsigned long long cum = incl - own;
    int dig = 7;
#pragma unroll
    for (int k = 7; k >= 0; --k) {                                // first k with cum + c[0..k] >= r
      unsigned long long pre = cum;
#pragma unroll
      for (int j = 0; j < k; ++j) pre += c[j];
      if (pre + c[k] >= r) dig = k;
    }
    unsigned long long before = cum;
    for (int j = 0; j < dig; ++j) before += c[j];
    const int digit = __shfl_sync(0xffffffffu, lane * 8 + dig, src);
    const unsigned long long bef = __shfl_sync(0xffffffffu, before, src);
    if (lane == 0) rank[i] = r - bef;
    pf = (pf << dp.width) | (unsigned long long)digit;
  }
  if (lane == 0) {
    prefix[i] = pf;
    if (d == 0) out[i] = counts[i / n_pct] ? (int64_t)(pf ^ kSign) : -1;
  }
}

// ---- fused latency statistics (ds_latency_stats): the percentiles of e2e / queue delay per (group, tier) and per
// group straight from start/done ticks. Nothing is materialised: every radix pass recomputes value = tick - arrival
// (8 B per request from HBM; arrival and tier are shared by the instances of a trace and stay in L2), and each value is
// counted in two segments: 3*g+tier ("tier" block, 3*G segments) and 3*G+g ("all" block, G segments).
struct LatArgs {
  const int64_t* trace_off; const int64_t* arrival; const uint8_t* tier; const ds_instance* inst; const int64_t* out_off;
  const int64_t* arr_ov;   // nullable: per-instance arrival ticks (closed loop), indexed like ticks
  const int64_t* ticks; const int32_t* group; const int64_t* t_mid; long long n_inst; int n_groups;   // groups after phases
  // Staging (optional, the part of the workspace beyond the histograms): the count pass leaves the low 32 bits of every key
  // and its segment code 3*g+tier (255 = not counted) at the request's output index. When every key agrees on bits 32..63
  // (latencies below 2^32 ticks = 71 minutes) the digit passes stream these 5 bytes per request linearly - mostly out of
  // L2 - instead of recomputing tick - arrival per instance (16 B per request and three dependent header loads per
  // instance, which made a pass that matches nothing cost 100 us for 164 MB).
  unsigned int* skey; unsigned char* scode; long long cap;
};
__device__ __forceinline__ bool stage_usable(const LatArgs& a, const Ws* hdr) {
  return a.skey != nullptr && !hdr->nostage && vary_top(hdr->and_bits ^ hdr->or_bits) <= 32;
}

// which of a staged key's (segment, percentile) prefixes it matches: bit q = its (group, tier) segment, bit 8+q = the
// group's "all" segment. NP = n_pct when it is 1..4 (unrolled, no loop or index arithmetic per percentile), 0 = any.
template <int NP>
__device__ __forceinline__ unsigned match32(const unsigned* pfx32, unsigned s_t, unsigned s_a, unsigned hi, int n_pct) {
  unsigned mm = 0;
  if (NP == 2) {                               // the report's (50, 99): one 8-byte read per segment
    const uint2 pt = *reinterpret_cast<const uint2*>(pfx32 + 2 * s_t), pa = *reinterpret_cast<const uint2*>(pfx32 + 2 * s_a);
    mm = (hi == pt.x ? 1u : 0u) | (hi == pt.y ? 2u : 0u) | (hi == pa.x ? 256u : 0u) | (hi == pa.y ? 512u : 0u);
  } else if (NP > 0) {
#pragma unroll
    for (int q = 0; q < NP; ++q) {
      mm |= (hi == pfx32[s_t * NP + q]) ? (1u << q) : 0u;
      mm |= (hi == pfx32[s_a * NP + q]) ? (256u << q) : 0u;
    }
  } else {
    for (int q = 0; q < n_pct; ++q) {
      mm |= (hi == pfx32[s_t * n_pct + q]) ? (1u << q) : 0u;
      mm |= (hi == pfx32[s_a * n_pct + q]) ? (256u << q) : 0u;
    }
  }
  return mm;
}

// kCount: segment counts + AND/OR of all keys. Otherwise: digit-d histogram of the keys matching each (segment, pct) prefix.
template <bool kCount>
__global__ void __launch_bounds__(1024) lat_pass_kernel(const LatArgs a, int n_pct, int d, Ws* hdr, unsigned long long* counts,
                                                       const unsigned long long* __restrict__ prefix, unsigned int* hist) {
  extern __shared__ unsigned int sh[];
  const int n_seg = 4 * a.n_groups;
  const int nb = kCount ? n_seg : n_seg * n_pct * 256;
  DigitPos dp; dp.lo = 0; dp.width = 0; dp.active = true;
  if (!kCount) {
    dp = digit_pos(hdr->and_bits ^ hdr->or_bits, 7 - d);
    if (!hdr->any || !dp.active) return;                           // no varying bits left for this pass
  }
  for (int i = threadIdx.x; i < nb; i += blockDim.x) sh[i] = 0;
  __shared__ unsigned long long pfx_s[kMaxSegPct];                  // the prefixes, read 2 x n_pct times per key
  __shared__ __align__(8) unsigned int pfx32_s[kMaxSegPct];                      // staged passes: bits [hshift, 32) of the prefixes
  if (!kCount) {
    const int hs = dp.lo + dp.width;
    for (int i = threadIdx.x; i < n_seg * n_pct; i += blockDim.x) {
      const unsigned long long pf = prefix[i];
      pfx_s[i] = pf;
      pfx32_s[i] = hs >= 32 ? 0u : ((unsigned)pf & (0xffffffffu >> hs));
    }
  }
  __syncthreads();
  unsigned long long kand = ~0ull, kor = 0ull; bool any = false;
  const int shift = dp.lo, hshift = dp.lo + dp.width;
  const unsigned dmask = (1u << dp.width) - 1u;
  // First digit pass: every prefix still is the bits common to ALL keys, so each key matches all of its (segment,
  // percentile) pairs. Only the (group, tier) histogram of percentile 0 is built from the keys; the group's "all"
  // histogram (the sum over its tiers) and the other percentiles' copies are filled in shared memory afterwards:
  // one add per key instead of 2 x n_pct. The count pass does the same with the segment counts.
  const bool first = !kCount && d == 7;
  // one WARP per instance: the dependent header loads (instance -> trace -> offsets) of 16 warps per block overlap
  const int lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
  bool stage = a.skey != nullptr;      // count pass: this warp may still write staged keys
  if (!kCount && stage_usable(a, hdr)) {
    // staged pass, all in 32 bits (measured: the 64-bit form of this loop - variable 64-bit shifts, 8-byte prefix compares -
    // executed 120 instructions per key and was issue-bound at 80-110 us for 102 MB). Every key agrees with every prefix
    // on bits 32..63 (they are common to all keys), so only bits [hshift, 32) are compared.
    // kKeys consecutive requests per thread and trip (16-byte key loads + 4-byte code loads, all issued before the first use:
    // the bytes in flight per SM, not the arithmetic, set the speed of these passes), the grid strides over the requests.
    const long long n = a.out_off[a.n_inst];
    const unsigned segall0 = 3u * (unsigned)a.n_groups;
    constexpr int kKeys = DS_K3_KEYS;
    const long long gstride = (long long)gridDim.x * blockDim.x * kKeys, nr = (n + 32 * kKeys - 1) / (32 * kKeys) * (32 * kKeys);   // warp-uniform trips
    auto run = [&](auto np_tag, auto first_tag) {
      constexpr int NP = decltype(np_tag)::value;
      constexpr bool kFirst = decltype(first_tag)::value;
      for (long long i4 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * kKeys; i4 < nr; i4 += gstride) {
        unsigned kk[kKeys], cc[kKeys];
        if (i4 + kKeys - 1 < n) {
#pragma unroll
          for (int v = 0; v < kKeys / 4; ++v) {
            const uint4 kv = *reinterpret_cast<const uint4*>(a.skey + i4 + 4 * v);
            const uchar4 cv = *reinterpret_cast<const uchar4*>(a.scode + i4 + 4 * v);
            kk[4 * v] = kv.x; kk[4 * v + 1] = kv.y; kk[4 * v + 2] = kv.z; kk[4 * v + 3] = kv.w;
            cc[4 * v] = cv.x; cc[4 * v + 1] = cv.y; cc[4 * v + 2] = cv.z; cc[4 * v + 3] = cv.w;
          }
        } else {
#pragma unroll
          for (int u = 0; u < kKeys; ++u) { const bool in = i4 + u < n; kk[u] = in ? a.skey[i4 + u] : 0u; cc[u] = in ? a.scode[i4 + u] : 255u; }
        }
#pragma unroll
        for (int u = 0; u < kKeys; ++u) {
          const bool ok = cc[u] != 255u;
          const unsigned s_t = ok ? cc[u] : 0u;
          if (kFirst) {    // every key matches every prefix of its segments: one add, the other histograms follow from it
            hist_add(sh, ok, (s_t * n_pct) * 256 + ((kk[u] >> shift) & dmask));
            continue;
          }
          const unsigned hi = __funnelshift_r(kk[u], 0u, hshift);                     // kk >> hshift, 0 when hshift = 32
          const unsigned s_a = segall0 + ((s_t * 171u) >> 9);                          // x/3 for x < 256
          if (NP == 2) {   // reject first with one predicate (four chained compares), build the match mask only for survivors
            const uint2 pt = *reinterpret_cast<const uint2*>(pfx32_s + 2 * s_t), pa = *reinterpret_cast<const uint2*>(pfx32_s + 2 * s_a);
            const bool hit = ok & ((hi == pt.x) | (hi == pt.y) | (hi == pa.x) | (hi == pa.y));
            if (!__any_sync(0xffffffffu, hit)) continue;
          }
          const unsigned mm = ok ? match32<NP>(pfx32_s, s_t, s_a, hi, n_pct) : 0u;
          const unsigned dig = (kk[u] >> shift) & dmask;
          if (mm) {                              // plain atomics by the matching lanes (see hist_add)
            for (int q = 0; q < n_pct; ++q) {
              if ((mm >> q) & 1u) atomicAdd(&sh[(s_t * n_pct + q) * 256 + dig], 1u);
              if ((mm >> (8 + q)) & 1u) atomicAdd(&sh[(s_a * n_pct + q) * 256 + dig], 1u);
            }
          }
        }
      }
    };
    if (first) run(std::integral_constant<int, 0>{}, std::true_type{});
    else if (n_pct == 2) run(std::integral_constant<int, 2>{}, std::false_type{});
    else if (n_pct == 1) run(std::integral_constant<int, 1>{}, std::false_type{});
    else if (n_pct == 3) run(std::integral_constant<int, 3>{}, std::false_type{});
    else run(std::integral_constant<int, 0>{}, std::false_type{});
  } else
  for (long long ii = (long long)blockIdx.x * nwarp + (threadIdx.x >> 5); ii < a.n_inst; ii += (long long)gridDim.x * nwarp) {
    const int t = a.inst[ii].trace;
    const long long lo = a.trace_off[t], n = a.trace_off[t + 1] - lo, oo = a.out_off[ii];
    const int g0 = a.group ? a.group[ii] : 0;
    const bool ph = a.t_mid != nullptr;
    const long long tm = ph ? a.t_mid[t] : 0;
    const bool gok = g0 >= 0 && (ph ? 2 * g0 + 1 : g0) < a.n_groups;
    if (kCount && stage) {
      // the staged passes walk [0, out_off[n_inst]) linearly: the instances' ranges must tile it in order; slots that no
      // request owns (padding between ranges, before the first one) are marked "not counted"
      const long long oe = a.out_off[ii + 1], gb = ii == 0 ? 0 : oo;
      if (oo < 0 || oe < oo + n || oe > a.cap) { if (lane == 0) atomicOr(&hdr->nostage, 1u); stage = false; }
      else {
        for (long long j = gb + lane; j < oo; j += 32) a.scode[j] = 255;
        for (long long j = oo + n + lane; j < oe; j += 32) a.scode[j] = 255;
      }
    }
    const int64_t* __restrict__ ap = a.arr_ov ? a.arr_ov + oo : a.arrival + lo;
    for (long long base = 0; base < n; base += 32 * kUnroll) {   // warp-uniform trip count
      long long av[kUnroll], tv[kUnroll]; int tr[kUnroll];
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        const long long r = base + u * 32 + lane;
        const bool in = r < n;
        av[u] = in ? ap[r] : 0; tv[u] = in ? a.ticks[oo + r] : 0; tr[u] = in ? (int)a.tier[lo + r] : -1;
      }
#pragma unroll
      for (int u = 0; u < kUnroll; ++u) {
        const bool ok = gok && tr[u] >= 0 && tr[u] <= 2;
        const unsigned long long k = (unsigned long long)(tv[u] - av[u]) ^ kSign;
        const int g = !ok ? 0 : (ph ? g0 * 2 + (av[u] >= tm ? 1 : 0) : g0);
        const unsigned s_t = (unsigned)(3 * g + (ok ? tr[u] : 0)), s_a = (unsigned)(3 * a.n_groups + g);
        if (kCount) {
          if (ok) { kand &= k; kor |= k; any = true; }
          hist_add(sh, ok, s_t);                   // (s_a's count is the sum over the group's tiers: added after the loop)
          const long long r = base + u * 32 + lane;
          if (stage && r < n) { a.skey[oo + r] = (unsigned)k; a.scode[oo + r] = ok ? (unsigned char)s_t : (unsigned char)255; }
        } else {
          const unsigned long long hi = hshift >= 64 ? 0ull : (k >> hshift);
          const unsigned dig = (unsigned)(k >> shift) & dmask;
          if (first) { hist_add(sh, ok, (s_t * n_pct) * 256 + dig); continue; }
          // which of the key's (segment, percentile) prefixes it matches: bit q = tier segment, bit 8+q = "all" segment.
          // After the first pass almost no key matches anything: one vote rejects the whole warp.
          unsigned mm = 0;
          for (int q = 0; q < n_pct; ++q) {
            mm |= (ok && hi == pfx_s[s_t * n_pct + q]) ? (1u << q) : 0u;
            mm |= (ok && hi == pfx_s[s_a * n_pct + q]) ? (256u << q) : 0u;
          }
          if (mm) {                              // plain atomics, see the staged loop
            for (int q = 0; q < n_pct; ++q) {
              if ((mm >> q) & 1u) atomicAdd(&sh[(s_t * n_pct + q) * 256 + dig], 1u);
              if ((mm >> (8 + q)) & 1u) atomicAdd(&sh[(s_a * n_pct + q) * 256 + dig], 1u);
            }
          }
        }
      }
    }
  }
  __syncthreads();
  if (kCount) {
    for (int g = threadIdx.x; g < a.n_groups; g += blockDim.x) sh[3 * a.n_groups + g] = sh[3 * g] + sh[3 * g + 1] + sh[3 * g + 2];
    __syncthreads();
  } else if (first) {
    for (int i = threadIdx.x; i < a.n_groups * 256; i += blockDim.x) {
      const int g = i >> 8, dg = i & 255;
      unsigned sum = 0;
      for (int t = 0; t < 3; ++t) {
        const unsigned c = sh[((3 * g + t) * n_pct) * 256 + dg];
        sum += c;
        for (int q = 1; q < n_pct; ++q) sh[((3 * g + t) * n_pct + q) * 256 + dg] = c;
      }
      for (int q = 0; q < n_pct; ++q) sh[((3 * a.n_groups + g) * n_pct + q) * 256 + dg] = sum;
    }
    __syncthreads();
  }
  if (kCount) {
    for (int dd = 16; dd > 0; dd >>= 1) { kand &= __shfl_xor_sync(0xffffffffu, kand, dd); kor |= __shfl_xor_sync(0xffffffffu, kor, dd); }
    const unsigned anym = __ballot_sync(0xffffffffu, any);
    if ((threadIdx.x & 31) == 0 && anym) { atomicAnd(&hdr->and_bits, kand); atomicOr(&hdr->or_bits, kor); atomicOr(&hdr->any, 1u); }
    for (int i = threadIdx.x; i < nb; i += blockDim.x) if (sh[i]) atomicAdd(&counts[i], (unsigned long long)sh[i]);
  } else {
    for (int i = threadIdx.x; i < nb; i += blockDim.x) if (sh[i]) atomicAdd(&hist[i], sh[i]);
  }
}

}  // namespace k3

size_t ws_tail_stats(int64_t n_seg, int64_t n_pct) { return k3::make_layout(nullptr, n_seg, n_pct).total; }
// staging area of ds_latency_stats for n_total simulated requests: u32 keys | u8 segment codes
size_t ws_latency_stage(int64_t n_total) { return n_total > 0 ? align_up(5 * (size_t)n_total, 256) + 1024 : 0; }   // (the callee keeps 512 for alignment)

}  // namespace ds

extern "C" int ds_latencies(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off, int64_t n_total,
                            const int64_t* arrival_override, const int64_t* start_tick, const int64_t* done_tick, const int32_t* group, const int64_t* t_mid,
                            int64_t* e2e, int64_t* qdelay, int32_t* seg_tier, int32_t* seg_all, void* stream) {
  using namespace ds;
  if (!tr || n_inst < 0 || n_total < 0) return DS_EINVAL;
  if (n_inst == 0 || n_total == 0) return DS_OK;
  if (!inst || !out_off || !start_tick || !done_tick || !e2e || !qdelay || n_inst > 0x7fffffff) return DS_EINVAL;
  k3::latencies_kernel<<<(unsigned)n_inst, 256, 0, (cudaStream_t)stream>>>(tr->trace_off, tr->arrival_tick, tr->tier, inst, out_off,
                                                                        arrival_override, start_tick, done_tick, group, t_mid, e2e, qdelay, seg_tier, seg_all);
  note_launch();
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}

extern "C" int ds_tail_stats(const int64_t* values, const int32_t* seg_id, int64_t n, int32_t n_segments, const int32_t* pct,
                             int32_t n_pct, int64_t* out, int64_t* count_out, void* workspace, size_t workspace_bytes, void* stream) {
  using namespace ds;
  if (n < 0 || n_segments < 1 || n_pct < 1 || n_pct > k3::kMaxPct || !pct || !out || !workspace) return DS_EINVAL;
  if (n > 0 && (!values || !seg_id)) return DS_EINVAL;
  if (n >= (1ll << 32) || (long long)n_segments * n_pct > (1 << 22)) return DS_EINVAL;
  k3::Pcts pc;
  for (int q = 0; q < n_pct; ++q) { if (pct[q] < 0 || pct[q] > 100) return DS_EINVAL; pc.p[q] = pct[q]; }
  k3::Layout L = k3::make_layout(workspace, n_segments, n_pct);
  if (workspace_bytes < L.total) return DS_ENOMEM;
  cudaStream_t s = (cudaStream_t)stream;
  DS_CUDA(cudaMemsetAsync(workspace, 0, L.total, s));
  DS_CUDA(cudaMemsetAsync(&L.hdr->and_bits, 0xff, 8, s));
  const int nsq = n_segments * n_pct;
  const int threads = 512;
  long long blocks = (n + threads * k3::kUnroll - 1) / (threads * k3::kUnroll);
  if (blocks > num_sms() * 4) blocks = num_sms() * 4;
  if (blocks < 1) blocks = 1;
  const size_t csm = n_segments <= 4096 ? sizeof(unsigned) * (size_t)n_segments : 0;
  k3::count_kernel<<<(unsigned)blocks, threads, csm, s>>>(values, seg_id, n, n_segments, L.hdr, L.counts);
  k3::init_kernel<<<(nsq + 255) / 256, 256, 0, s>>>(L.counts, n_segments, n_pct, pc, L.hdr, L.prefix, L.rank, count_out);
  note_launch(2);
  const size_t hsm = sizeof(unsigned) * 256 * (size_t)nsq;
  const bool priv = hsm <= 160 * 1024;
  if (priv && attr_needed(DS_ATTR_K3_HIST))
    DS_CUDA(cudaFuncSetAttribute(k3::hist_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024));
  long long per_sm = priv ? (long long)(200 * 1024) / (long long)(hsm + 1024) : 4;   // resident blocks by shared memory
  if (per_sm > 4) per_sm = 4;
  if (per_sm < 1) per_sm = 1;
  long long hblocks = priv ? (long long)num_sms() * per_sm : blocks;
  if (hblocks > blocks) hblocks = blocks;
  for (int d = 7; d >= 0; --d) {
    if (priv) k3::hist_kernel<true><<<(unsigned)hblocks, threads, hsm, s>>>(values, seg_id, n, n_segments, n_pct, d, L.hdr, L.prefix, L.hist);
    else k3::hist_kernel<false><<<(unsigned)blocks, threads, 0, s>>>(values, seg_id, n, n_segments, n_pct, d, L.hdr, L.prefix, L.hist);
    k3::select_kernel<<<(nsq + 3) / 4, 128, 0, s>>>(n_segments, n_pct, d, L.hdr, L.counts, L.prefix, L.rank, L.hist, out);
    note_launch(2);
  }
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}

extern "C" int ds_latency_stats(const ds_traces* tr, const ds_instance* inst, int64_t n_inst, const int64_t* out_off,
                                const int64_t* arrival_override, const int64_t* start_tick, const int64_t* done_tick, const int32_t* group, int32_t n_groups,
                                const int64_t* t_mid, const int32_t* pct, int32_t n_pct, int64_t* e2e_out, int64_t* qdelay_out,
                                int64_t* count_out, void* workspace, size_t workspace_bytes, void* stream) {
  using namespace ds;
  if (!tr || n_inst < 0 || n_groups < 1 || n_pct < 1 || n_pct > k3::kMaxPct || !pct || !workspace) return DS_EINVAL;
  if (!e2e_out && !qdelay_out) return DS_EINVAL;
  if (n_inst > 0 && (!inst || !out_off || !tr->trace_off || (!arrival_override && !tr->arrival_tick) || !tr->tier)) return DS_EINVAL;
  if ((e2e_out && !done_tick) || (qdelay_out && !start_tick)) { if (n_inst > 0) return DS_EINVAL; }
  const int G = n_groups * (t_mid ? 2 : 1), n_seg = 4 * G, nsq = n_seg * n_pct;
  const size_t hsm = sizeof(unsigned) * 256 * (size_t)nsq;
  if (hsm > 200 * 1024) return DS_EINVAL;   // (groups x phases x 4 x percentiles) histograms must fit shared memory
  k3::Pcts pc;
  for (int q = 0; q < n_pct; ++q) { if (pct[q] < 0 || pct[q] > 100) return DS_EINVAL; pc.p[q] = pct[q]; }
  k3::Layout L = k3::make_layout(workspace, n_seg, n_pct);
  if (workspace_bytes < L.total) return DS_ENOMEM;
  cudaStream_t s = (cudaStream_t)stream;
  if (attr_needed(DS_ATTR_K3_LAT))
    DS_CUDA(cudaFuncSetAttribute(k3::lat_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024));
  long long per_sm = (long long)(200 * 1024) / (long long)(hsm + 1024);
  if (per_sm > 3) per_sm = 3;
  if (per_sm < 1) per_sm = 1;
  // when the histograms leave room for one block per SM only (configs[3]/[4]: 160 KB), that block runs 32 warps instead of 16
  const int threads = per_sm == 1 ? 1024 : 512;
  long long blocks = (long long)num_sms() * per_sm;
  if (blocks > (n_inst + threads / 32 - 1) / (threads / 32)) blocks = (n_inst + threads / 32 - 1) / (threads / 32);
  if (blocks < 1) blocks = 1;
  for (int metric = 0; metric < 2; ++metric) {
    int64_t* out = metric == 0 ? e2e_out : qdelay_out;
    if (!out) continue;
    DS_CUDA(cudaMemsetAsync(workspace, 0, L.total, s));
    DS_CUDA(cudaMemsetAsync(&L.hdr->and_bits, 0xff, 8, s));
    if (n_inst == 0) {   // all segments empty
      k3::init_kernel<<<(nsq + 255) / 256, 256, 0, s>>>(L.counts, n_seg, n_pct, pc, L.hdr, L.prefix, L.rank, count_out);
      k3::select_kernel<<<(nsq + 3) / 4, 128, 0, s>>>(n_seg, n_pct, 0, L.hdr, L.counts, L.prefix, L.rank, L.hist, out);
      note_launch(2);
      continue;
    }
    k3::LatArgs a{tr->trace_off, tr->arrival_tick, tr->tier, inst, out_off, arrival_override, metric == 0 ? done_tick : start_tick, group, t_mid,
                  (long long)n_inst, G, nullptr, nullptr, 0};
    // whatever the caller's workspace holds beyond the histograms is the staging area (5 bytes per simulated request)
    const size_t extra = workspace_bytes - L.total;
    if (extra >= 512 + 5) {
      long long cap = (long long)((extra - 512) / 5);
      if (cap > 0xffffffffll) cap = 0xffffffffll;
      a.cap = cap;
      a.skey = (unsigned int*)((char*)workspace + L.total);
      a.scode = (unsigned char*)workspace + L.total + align_up(4 * (size_t)cap, 256);
    }
    k3::lat_pass_kernel<true><<<(unsigned)blocks, threads, sizeof(unsigned) * (size_t)n_seg, s>>>(a, n_pct, 0, L.hdr, L.counts, L.prefix, L.hist);
    k3::init_kernel<<<(nsq + 255) / 256, 256, 0, s>>>(L.counts, n_seg, n_pct, pc, L.hdr, L.prefix, L.rank, count_out);
    note_launch(2);
    for (int d = 7; d >= 0; --d) {
      k3::lat_pass_kernel<false><<<(unsigned)blocks, threads, hsm, s>>>(a, n_pct, d, L.hdr, L.counts, L.prefix, L.hist);
      k3::select_kernel<<<(nsq + 3) / 4, 128, 0, s>>>(n_seg, n_pct, d, L.hdr, L.counts, L.prefix, L.rank, L.hist, out);
      note_launch(2);
    }
  }
  DS_CUDA(cudaGetLastError());
  return DS_OK;
}

// ---------------------------------------------------------------------------------------------------------------------
// ds_tail_stats_static: ds_tail_stats for callers that cannot allocate (code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc). The scratch that ds_tail_stats takes from its caller (header, segment counts,
// prefixes, ranks, radix histograms) lives in ONE file-scope device array of a fixed, modest size instead; the caller
// still passes inputs and outputs. The array exists on every GPU that loads the library, until the process exits.
//
// In HOST code the array's name is a host-side stand-in, not a device address: a kernel given `g_tail_scratch` itself
// would fault (or, where the GPU can reach host memory, silently use the wrong memory). The device address is looked up
// once per device, with that device current, by cudaGetSymbolAddress below, and only that pointer is handed on.
namespace ds {
namespace k3 {

constexpr int kStaticMaxSegPct = DS_TAIL_STATS_STATIC_MAX_SEGPCT;   // n_segments * n_pct (and n_segments) at most this
// the largest Layout (make_layout) any admitted (n_segments, n_pct) needs: header 256 + counts + prefix + rank (each
// 8 bytes per entry, rounded up to 256) + 256 32-bit bins per (segment, percentile)
constexpr size_t kStaticRow = (8 * (size_t)kStaticMaxSegPct + 255) / 256 * 256;
constexpr size_t kStaticBytes = 256 + 3 * kStaticRow + 4 * 256 * (size_t)kStaticMaxSegPct;   // 134 400 bytes at 128
static_assert(kStaticBytes == DS_TAIL_STATS_STATIC_BYTES, "the header states the size of the built-in scratch");
static __device__ __align__(256) unsigned char g_tail_scratch[kStaticBytes];

constexpr int kStaticMaxDevices = 64;
static unsigned char* g_tail_scratch_ptr[kStaticMaxDevices];   // device address of g_tail_scratch, per device (nullptr: not looked up yet)
static std::mutex g_tail_scratch_mu;

// device address of the scratch array on the calling thread's current device; nullptr (error recorded) on a CUDA error
static unsigned char* static_scratch() {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) { cuda_fail(e); return nullptr; }
  if (dev < 0 || dev >= kStaticMaxDevices) { cuda_fail(cudaErrorInvalidDevice); return nullptr; }
  std::lock_guard<std::mutex> lk(g_tail_scratch_mu);
  if (!g_tail_scratch_ptr[dev]) {
    unsigned char* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_tail_scratch);       // the set-up step: once per device, that device current
    if (e != cudaSuccess || !ptr) { cuda_fail(e != cudaSuccess ? e : cudaErrorInvalidSymbol); return nullptr; }
    g_tail_scratch_ptr[dev] = ptr;
  }
  return g_tail_scratch_ptr[dev];
}

}  // namespace k3
}  // namespace ds

extern "C" int ds_tail_stats_static(const int64_t* values, const int32_t* seg_id, int64_t n, int32_t n_segments, const int32_t* pct,
                                    int32_t n_pct, int64_t* out, int64_t* count_out, void* stream) {
  using namespace ds;
  if (n_segments < 1 || n_pct < 1 || n_pct > k3::kMaxPct) return DS_EINVAL;
  // beyond the built-in scratch: refuse, never spill (the caller can use ds_tail_stats with a workspace of its own)
  if (n_segments > k3::kStaticMaxSegPct || (long long)n_segments * n_pct > k3::kStaticMaxSegPct) return DS_ELIMIT;
  if (k3::make_layout(nullptr, n_segments, n_pct).total > k3::kStaticBytes) return DS_ELIMIT;   // (implied by the two tests above)
  unsigned char* ws = k3::static_scratch();
  if (!ws) return DS_ECUDA;
  // ds_tail_stats clears the whole layout (cudaMemsetAsync on `stream`) before its first kernel, so what the previous
  // call left in the shared array is never read. It launches kernels and memsets only: no cudaMalloc / cudaFree.
  return ds_tail_stats(values, seg_id, n, n_segments, pct, n_pct, out, count_out, ws, k3::kStaticBytes, stream);
}
