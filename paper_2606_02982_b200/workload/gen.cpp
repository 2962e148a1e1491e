// Seeded synthetic input generators (BASELINE.json:configs[0..4]).
//
// This module produces INPUT ARRAYS ONLY: packed prompt text + offsets, tiers, output lengths,
// unit-mean exponential inter-arrival draws, and (for the text-free configs 3/4) per-request
// (words, tokens) drawn from the distributions the text generator induces. It contains none of
// the method's arithmetic: no word/token counting of bytes, no estimate, no queue, no policy,
// no EMA, no percentile. Both the CPU oracle's tests and the CUDA path's tests/bench read the
// arrays written here; neither side's results ever flow back into this file.
//
// RNG: splitmix64 streams keyed by (seed, purpose, a, b); every prompt / request has its own
// stream, so generation is order-independent and parallel.
#include <cstdint>
#include <cmath>
#include <cstring>
#include <thread>
#include <vector>
#include <algorithm>

namespace {

typedef uint64_t u64;

inline u64 mix64(u64 z) {
  z += 0x9E3779B97F4A7C15ull;
  z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
  z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
  return z ^ (z >> 31);
}

struct Rng {
  u64 s;
  Rng(u64 seed, u64 purpose, u64 a, u64 b) {
    s = mix64(seed ^ 0xD1B54A32D192ED03ull);
    s = mix64(s ^ (purpose * 0x9E3779B97F4A7C15ull));
    s = mix64(s ^ (a * 0xC2B2AE3D27D4EB4Full));
    s = mix64(s ^ (b * 0x165667B19E3779F9ull));
  }
  inline u64 next() { s += 0x9E3779B97F4A7C15ull; u64 z = s;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull; z = (z ^ (z >> 27)) * 0x94D049BB133111EBull; return z ^ (z >> 31); }
  // uniform in (0,1): never 0, never 1
  inline double uni() { return ((double)(next() >> 11) + 0.5) * (1.0 / 9007199254740992.0); }
  inline uint32_t below(uint32_t n) { return (uint32_t)(((next() >> 32) * (u64)n) >> 32); }
  inline double normal() { double u1 = uni(), u2 = uni(); return std::sqrt(-2.0 * std::log(u1)) * std::cos(6.283185307179586476925 * u2); }
};

enum Purpose : u64 { P_TEXT = 1, P_REQ = 2, P_SCANLEN = 3, P_SCANTEXT = 4, P_NUMERIC = 5 };

const char kPunct[6] = {'.', ',', ';', ':', '!', '?'};
const char kSep[3] = {' ', '\t', '\n'};

struct WordLaw { double p_geo; double p_punct; };

// word length: min(12, Geometric_1(p)), support 1,2,...
inline int word_len(Rng& r, double p) {
  int L = 1;
  while (L < 12 && r.uni() >= p) ++L;
  return L;
}

template <class F> void parallel_for(int64_t n, int n_threads, F f) {
  if (n_threads <= 1 || n < 2) { f(0, n); return; }
  std::vector<std::thread> th;
  int64_t chunk = (n + n_threads - 1) / n_threads;
  for (int t = 0; t < n_threads; ++t) {
    int64_t a = t * chunk, b = std::min<int64_t>(n, a + chunk);
    if (a >= b) break;
    th.emplace_back([=] { f(a, b); });
  }
  for (auto& x : th) x.join();
}

// One cfg0/1-style prompt: n_words ~ U{5..200}; words of word_len letters a-z (+ one punct byte
// w.p. p_punct); separators between words: run length U{1,2,3} of {space,tab,newline}; none at
// the edges. If out==nullptr only the size is returned.
int64_t gen_prompt(u64 seed, u64 stream, u64 idx, WordLaw law, uint8_t* out) {
  Rng r(seed, P_TEXT, stream, idx);
  int n_words = 5 + (int)r.below(196);
  int64_t k = 0;
  for (int w = 0; w < n_words; ++w) {
    if (w) { int run = 1 + (int)r.below(3); for (int j = 0; j < run; ++j) { uint8_t c = (uint8_t)kSep[r.below(3)]; if (out) out[k] = c; ++k; } }
    int L = word_len(r, law.p_geo);
    for (int j = 0; j < L; ++j) { uint8_t c = (uint8_t)('a' + r.below(26)); if (out) out[k] = c; ++k; }
    if (r.uni() < law.p_punct) { uint8_t c = (uint8_t)kPunct[r.below(6)]; if (out) out[k] = c; ++k; }
  }
  return k;
}

// cfg2-style prompt body of exactly `len` bytes: optional leading separator run, words, separator
// runs of U{0..8} (0 merges two words), cut at len wherever it falls. kind: 0 normal, 1 all-separator.
void gen_scan_prompt(u64 seed, u64 idx, int64_t len, int kind, uint8_t* out) {
  Rng r(seed, P_SCANTEXT, idx, 0);
  int64_t k = 0;
  if (kind == 1) { while (k < len) out[k++] = (uint8_t)kSep[r.below(3)]; return; }
  bool lead = r.below(2) != 0;   // prompts may begin on a separator run
  bool first = true;
  while (k < len) {
    if (!first || lead) { int run = (int)r.below(9); for (int j = 0; j < run && k < len; ++j) out[k++] = (uint8_t)kSep[r.below(3)]; }
    first = false;
    int L = word_len(r, 0.3);
    for (int j = 0; j < L && k < len; ++j) out[k++] = (uint8_t)('a' + r.below(26));
    if (r.uni() < 0.1 && k < len) out[k++] = (uint8_t)kPunct[r.below(6)];
  }
}

}  // namespace

extern "C" {

// Text for n_traces*n_req prompts (trace-major). law of prompt i: post_drift && post_drift[i] ?
// (p1,punct1) : (p0,punct0). bytes==nullptr: only offsets[0..n] (offsets[0]=0) are written.
// Returns total bytes, or -1 if cap is too small.
int64_t dsgen_text(uint64_t seed, int64_t n_traces, int64_t n_req, double p0, double punct0, double p1, double punct1,
                   const uint8_t* post_drift, uint8_t* bytes, int64_t cap, int64_t* offsets, int n_threads) {
  int64_t n = n_traces * n_req;
  WordLaw l0{p0, punct0}, l1{p1, punct1};
  if (!bytes) {
    parallel_for(n, n_threads, [&](int64_t a, int64_t b) {
      for (int64_t i = a; i < b; ++i)
        offsets[i + 1] = gen_prompt(seed, (u64)(i / n_req), (u64)(i % n_req), (post_drift && post_drift[i]) ? l1 : l0, nullptr);
    });
    offsets[0] = 0;
    for (int64_t i = 0; i < n; ++i) offsets[i + 1] += offsets[i];
    return offsets[n];
  }
  if (offsets[n] > cap) return -1;
  parallel_for(n, n_threads, [&](int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i)
      gen_prompt(seed, (u64)(i / n_req), (u64)(i % n_req), (post_drift && post_drift[i]) ? l1 : l0, bytes + offsets[i]);
  });
  return offsets[n];
}

// Per-request draws shared by all trace configs. out_dist 0: clamp(round(LogNormal(4.5,0.8)),1,512);
// 1: min(4096, floor(16*U^(-1/1.5))). tier 20/50/30. expo = -ln(U) (unit-mean inter-arrival draw).
void dsgen_requests(uint64_t seed, int64_t n_traces, int64_t n_req, int out_dist,
                    uint8_t* tier, int32_t* out_len, double* expo, int n_threads) {
  int64_t n = n_traces * n_req;
  parallel_for(n, n_threads, [&](int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i) {
      Rng r(seed, P_REQ, (u64)(i / n_req), (u64)(i % n_req));
      double u = r.uni();
      tier[i] = u < 0.2 ? 0 : (u < 0.7 ? 1 : 2);
      if (out_dist == 0) {
        double v = std::exp(4.5 + 0.8 * r.normal());
        long long o = std::llround(v); if (o < 1) o = 1; if (o > 512) o = 512; out_len[i] = (int32_t)o;
      } else {
        double v = std::floor(16.0 * std::pow(r.uni(), -1.0 / 1.5)); if (v > 4096.0) v = 4096.0; out_len[i] = (int32_t)v;
      }
      expo[i] = -std::log(r.uni());
    }
  });
}

// Text-free (words, tokens) for configs 3/4: n_words ~ U{5..200}; each word contributes a token
// increment drawn from the categorical law the word generator induces (1 w.p. 1-q^4, 2 w.p.
// q^4-q^8, 3 w.p. q^8, q=1-p) plus one more w.p. p_punct. Distributionally identical to running
// the characterizer over dsgen_text output; tests compare the two on a materialised sample.
void dsgen_counts(uint64_t seed, int64_t n_traces, int64_t n_req, double p0, double punct0, double p1, double punct1,
                  const uint8_t* post_drift, int32_t* words, int32_t* tokens, int n_threads) {
  int64_t n = n_traces * n_req;
  parallel_for(n, n_threads, [&](int64_t a, int64_t b) {
    for (int64_t i = a; i < b; ++i) {
      bool post = post_drift && post_drift[i];
      double p = post ? p1 : p0, pp = post ? punct1 : punct0;
      double q4 = std::pow(1.0 - p, 4.0), q8 = q4 * q4;
      Rng r(seed, P_NUMERIC, (u64)(i / n_req), (u64)(i % n_req));
      int nw = 5 + (int)r.below(196);
      int t = 0;
      for (int w = 0; w < nw; ++w) {
        double u = r.uni();
        t += u < q8 ? 3 : (u < q4 ? 2 : 1);
        if (r.uni() < pp) ++t;
      }
      words[i] = nw; tokens[i] = t;
    }
  });
}

// cfg2 prompt lengths: min(65536, round(LogNormal(ln 600, 1.2))) bytes; ~1% forced empty, ~1%
// all-separator. Appends prompts until exactly total_bytes are used (last prompt truncated).
// Writes offsets[0..n] and kind[0..n) (0 normal, 1 all-separator); returns n (<= cap_prompts) or -1.
int64_t dsgen_scan_layout(uint64_t seed, int64_t total_bytes, int64_t cap_prompts, int64_t* offsets, uint8_t* kind) {
  int64_t pos = 0, n = 0;
  offsets[0] = 0;
  while (pos < total_bytes) {
    if (n >= cap_prompts) return -1;
    Rng r(seed, P_SCANLEN, (u64)n, 0);
    double u = r.uni();
    int64_t len; uint8_t kd = 0;
    if (u < 0.01) len = 0;
    else {
      if (u < 0.02) kd = 1;
      double v = std::exp(std::log(600.0) + 1.2 * r.normal());
      len = (int64_t)std::llround(v); if (len > 65536) len = 65536; if (len < 0) len = 0;
    }
    if (pos + len > total_bytes) len = total_bytes - pos;
    pos += len; kind[n] = kd; offsets[++n] = pos;
  }
  return n;
}

void dsgen_scan_fill(uint64_t seed, int64_t n_prompts, const int64_t* offsets, const uint8_t* kind,
                     int64_t first_prompt, int64_t end_prompt, uint8_t* bytes /*base of prompt first_prompt*/, int n_threads) {
  (void)n_prompts;
  int64_t base = offsets[first_prompt];
  parallel_for(end_prompt - first_prompt, n_threads, [&](int64_t a, int64_t b) {
    for (int64_t j = a; j < b; ++j) {
      int64_t i = first_prompt + j;
      gen_scan_prompt(seed, (u64)i, offsets[i + 1] - offsets[i], kind[i], bytes + (offsets[i] - base));
    }
  });
}

}  // extern "C"
