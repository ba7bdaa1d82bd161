// SciFi Seeding kernel (section 3) for sm_100a.
//
// One CTA per event-half (L372): the half's twelve sorted hit zones are staged into shared memory and stay
// there for every step (L370).  In the staged tile every zone is framed by a -inf and a +inf sentinel, so
// that no search needs a bounds check.  Stages, separated by __syncthreads():
//   S0  staging + bin tables           per zone, a 256-bin table "first hit with bin >= k" turns every lower
//                                      bound into one lookup plus a short forward scan (about 0.5 hits per
//                                      bin); the table is built by marking the first hit of every occupied
//                                      bin and a ballot-based suffix fill, one warp per zone
//   S1  two-hit + three-hit search     per iteration: thread per T1 hit finds its T3 window (Eq. 8-11) and
//                                      cuts it into items of at most 4 consecutive T3 hits; thread per item:
//                                      Eq. 3-5 and the T2 band (Eq. 12-13, A3/A4) for its pairs, with one
//                                      T2 pointer that only moves forward (the band moves monotonically with
//                                      x3); the triplets of both iterations go to one queue in shared memory
//   S2  extension                      thread per queued triplet: exact parabola, +-1 mm closest hit in
//                                      the other three x-layers, >= 5 hits -> queued candidate (L90)
//   S2b fit                            dense pass over the candidates: fixed-matrix least squares, chi2 cut
//   S3  clone kill                     64-bit atomicMin table per x-hit, vote pass (L183-200, Eq. 15);
//                                      survivors are compacted to the bottom of the work region
//   S4  u/v addition, iterative        (survivor, pass, first-layer hit) items (Eq. 16): phase A
//                                      walks three stereo layers of every item, phase B finishes the walks
//                                      that can still succeed
//   S4h u/v addition, Hough clusters   (lhcb_set_uv_hough, L217, reading A20) votes as 64-bit masks per
//                                      (survivor, layer), bit-sliced populations, hypothesis pass
//   S5  y fit + seed output            thread per queued combination: y fit, best per survivor by
//                                      packed-key atomicMin, the winner writes the seed
//
// Arithmetic: every formula follows DESIGN.md "Arithmetic specification" operation by operation;
// this translation unit is compiled with -fmad=false so that no multiply-add is contracted.
#pragma once
#include <cstdint>

#include "../../include/lhcb.h"

namespace lhcb {

#ifndef LHCB_LUT_BINS
#define LHCB_LUT_BINS 256
#endif
#ifndef LHCB_ITEM_PAIRS
#define LHCB_ITEM_PAIRS 4   // T3 hits per item of the pair walk (2, 4 or 8; measured 3.10 ms with 4 against 3.16 ms with 8)
#endif
constexpr int kSeedThreadsMax = 512;          // the kernel is instantiated for 256 x 5, 256 x 4 and 512 x 2 CTAs/SM
constexpr int kLutBins = LHCB_LUT_BINS;       // bins of the per-zone search table
constexpr int kItemPairs = LHCB_ITEM_PAIRS;
constexpr int kTileIndexBits = 13;            // tile indices fit 13 bits: max_hits_per_half + 40 <= 8192
constexpr unsigned long long kNoKey = ~0ull;
static_assert(kLutBins % 32 == 0, "the suffix fill of the bin tables works on whole warps of bins");
static_assert(kItemPairs == 2 || kItemPairs == 4 || kItemPairs == 8, "item length");

// Optional per-stage cycle counters (diagnostic build only: -DLHCB_STAGE_CLOCKS, bench.py --stage-clocks).
// Thread 0 of every CTA adds the cycles since its previous mark to g_stage_clk[i];
// lhcb_debug_stage_clocks() reads them.
#ifdef LHCB_STAGE_CLOCKS
__device__ unsigned long long g_stage_clk[16];
__device__ unsigned int g_dbg_max[8];     // maxima over CTAs: triplets, candidates, survivors, queued u/v combinations, ...
#define LHCB_DBG_MAX(i, v) if (threadIdx.x == 0) atomicMax(&g_dbg_max[i], (unsigned int)(v));
#define LHCB_CLK_INIT long long clk_prev__ = clock64();
#define LHCB_CLK(i)                                                                         \
  if (threadIdx.x == 0) {                                                                   \
    const long long t__ = clock64();                                                        \
    atomicAdd(&g_stage_clk[i], (unsigned long long)(t__ - clk_prev__));                     \
    clk_prev__ = t__;                                                                       \
  }
#else
#define LHCB_CLK_INIT
#define LHCB_CLK(i)
#define LHCB_DBG_MAX(i, v)
#endif

// Optional index checks (diagnostic build only: -DLHCB_CHECKED, tests/test_gpu_checked.py; compute-sanitizer is
// closed on the GPU pool).  LHCB_CHECK_IDX(i, n) records an index outside
// [0, n) in g_check = {failures, line of the first one, its index, its bound} and counts the checks made in
// g_check_count; lhcb_debug_checks() reads them.  The release build compiles the checks away.
#ifdef LHCB_CHECKED
__device__ unsigned int g_check[4];
__device__ unsigned long long g_check_count;
__device__ __noinline__ void check_fail(int line, long long i, long long n) {
  if (atomicAdd(&g_check[0], 1u) == 0u) { g_check[1] = (unsigned)line; g_check[2] = (unsigned)i; g_check[3] = (unsigned)n; }
}
#define LHCB_CHECK_IDX(i, n)                                                                          \
  do {                                                                                                \
    atomicAdd(&lhcb::g_check_count, 1ull);                                                            \
    if ((unsigned long long)(long long)(i) >= (unsigned long long)(long long)(n))                     \
      lhcb::check_fail(__LINE__, (long long)(i), (long long)(n));                                     \
  } while (0)
#else
#define LHCB_CHECK_IDX(i, n)
#endif

struct SeedParams {
  float zb[12], gz[12], tan_a[12], inv_tan[12], inv_z[12], zt[12];
  float ywin_a[2][12], ywin_b[2][12];
  int xl[6], ul[6], slot_of_layer[12];
  int l1[2], l2[2], l3[2];
  int ol[2][3], os[2][3], ss[2][3];   // per iteration: the three other x-layers, their x-slots, the x-slots of l1 l2 l3
  float dx3max[2], r13[2], inv_dz13[2], z1[2], dz12[2], K[2], inv_K[2], G13[2];
  float a, b, kappa, inv_kappa, f_lo, f_hi, d_lo, d_hi, tol_x, tol_uv, chi2x_max, chi2y_max;
  float wx[7], wy[7];
  float zbS, gS, gpS;
  int min_x_hits, min_uv_hits, uv_first[2], polarity;
  int max_seeds, max_cand, max_hits, max_trip;
  int uv_hough;                       // Hough-cluster UV seeding (L217, reading A20) instead of the iterative one
  float h_tlo[2], h_w, h_invw;        // its t_y bins: b = clamp((t - tlo[half]) * invw, 0, 63), width w
  int smem_total;   // dynamic shared memory of the launch = seed_smem_bytes(capacities)
  const float* P;   // [7][3][6]
  const float* Q;   // [64][2][6]
  // batch
  int n_events;
  uint32_t n_hits;
  const uint32_t* zone_off;
  const float* hit_x;
  const int8_t* pol;
  const uint32_t* order;   // optional CTA -> event-half map (heaviest halves first) or NULL
  uint32_t* done;          // optional per-half flags (workspace of lhcb_order): 0 while the half is being seeded, 1 when its
                           // seeds are in global memory; lets the Matching start before the whole Seeding grid has drained
  uint32_t* count;
  float* state;
  float* par;
  uint32_t* hits;
  uint8_t* nx;
  uint8_t* nuv;
  uint32_t* status;
  size_t cap_total;
};

// all hit references inside the kernel are TILE indices (position in the staged, sentinel-framed tile)
// a queued three-hit combination: zone-local indices of its hits in 10 bits each (a zone holds at most 1,023
// hits, else the half is reported as LHCB_ST_HITS_OVERFLOW) and the iteration: i1 | i2 << 10 | i3 << 20 | it << 30
typedef uint32_t Triplet;
constexpr int kZoneIndexBits = 10;
struct __align__(16) Cand { float ax, bx, cx, chi2; uint16_t hit[6]; uint8_t nx, it, keep, pattern; };   // nx = 0: rejected by the fit

struct __align__(16) Zone { int b, e; float x0, invw; };   // hits [b, e) of the tile; one 16-byte shared-memory load

struct SeedSmemHeader {
  unsigned long long mbar;
  unsigned long long pad_;
  Zone zi[12];         // per zone: [b, e) in the tile and bin(v) = clamp((v - x0) * invw, 0, kLutBins-1)
  float4 uvc[6];       // per stereo slot: {z tan(alpha), 1/tan(alpha), 1/z, layer index (int bits)}
  uint32_t zg[12];     // global hit index = tile index + zg[layer]
  int xoff[6];         // clone-table index of an x-hit = tile index + xoff[x-slot]
  int n_xhits;
  int n_trip, n_cand, n_kept, n_seed, n_live;
  unsigned int status;
  int warp_sums[2][kSeedThreadsMax / 32 + 1];   // two buffers: consecutive block scans never share one
};

constexpr int kSeedHeaderBytes = 640;
static_assert(sizeof(SeedSmemHeader) <= kSeedHeaderBytes, "shared-memory header overflows its slot");

// Shared-memory map of one CTA, all offsets 16-byte aligned:
//   [header | bin tables | kept list u16[max_cand] | hits tile (the half's ACTUAL size) | work region W ... |
//    x-z candidates, filled downward from the end]
// The tile holds, per zone, [..., -inf, hits ..., +inf, ...].  W holds the triplet queue, then the clone table, then the
// u/v queues; it starts right after the tile and ends where the candidates begin, so a half with fewer hits or
// candidates than the capacities leaves more room for the queues.  The capacities guarantee
// W >= max_trip * 4 bytes (seed_w_bytes).  During S1 the (still empty) candidate slots hold the items of the pair walk.
__host__ __device__ inline size_t seed_align16(size_t b) { return (b + 15) & ~(size_t)15; }
__host__ __device__ inline size_t seed_off_kept() { return kSeedHeaderBytes + seed_align16(12 * (kLutBins + 1) * 2); }
__host__ __device__ inline size_t seed_off_hits(int max_cand) { return seed_off_kept() + seed_align16((size_t)max_cand * 2); }
// tile: per zone [-inf, -inf, hits ..., +inf]
__host__ __device__ inline size_t seed_tile_bytes(int n_hits) { return seed_align16(((size_t)n_hits + 36) * 4 + 16); }
// W minimum: the triplet queue.  (The clone table, 8 bytes per x-hit, takes W plus the candidate slots that are
// still free when the clone kill starts; a half whose table does not fit is reported, LHCB_ST_HITS_OVERFLOW.)
// W and the candidate slots together also hold the staging buffer of S0 (the half's hits before they move into the tile).
__host__ __device__ inline size_t seed_w_bytes(int max_hits, int max_cand, int max_trip) {
  const size_t q = (size_t)max_trip * sizeof(Triplet), stg = ((size_t)max_hits + 8) * 4, c = (size_t)max_cand * 32;
  return seed_align16(stg > q + c ? stg - c : q);
}
__host__ __device__ inline size_t seed_smem_bytes(int max_hits, int max_cand, int max_trip) {
  size_t b = seed_off_hits(max_cand);
  b += seed_tile_bytes(max_hits);                           // hits tile with its sentinels
  b += seed_w_bytes(max_hits, max_cand, max_trip);         // work region W (minimum)
  b += (size_t)max_cand * 32;                              // candidates
  return b;
}

// ------------------------------------------------------------------------------------ searches
// Sorted zone framed by sentinels + bin table.  lut[k] = first tile index whose bin is >= k
// (lut[kLutBins] = zone end, the +inf sentinel).  bin() is monotone in v, so every hit before lut[bin(v)] is
// < v: the exact lower/upper bound is lut[bin(v)] plus a forward scan inside one bin (about half a hit per
// bin), which the +inf sentinel ends.  Pure comparisons: the result is identical to a binary search, whatever
// the rounding of bin().
// bin(v): any monotone function of v used alike by the table build and the lookups.  Rounded to the nearest
// integer by adding 2^23 (one FADD instead of a conversion on the slower XU pipe); NaN lands in bin 0.
__device__ __forceinline__ int zone_bin(const Zone& z, float v) {
  float t = (v - z.x0) * z.invw;
  t = fminf(fmaxf(t, 0.f), (float)(kLutBins - 1));
  const int k = __float_as_int(t + 8388608.f) & 0x3FF;
  LHCB_CHECK_IDX(k, kLutBins);
  return k;
}
static_assert(kLutBins <= 1024, "zone_bin keeps ten bits");

// shared-memory counter + 1, returning the old value: one ATOMS per lane (the compiler's warp-aggregated
// atomicAdd costs about twenty instructions on the divergent paths where the queues are appended)
__device__ __forceinline__ int smem_inc(int* counter) {
  int old;
  asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(old) : "r"((uint32_t)__cvta_generic_to_shared(counter)) : "memory");
  return old;
}
// first index in [b, e] with x[i] >= v, also returning x[i] (+inf at e)
__device__ __forceinline__ int lower_bound_v(const float* __restrict__ x, const uint16_t* __restrict__ lut,
                                             const Zone& z, float v, float& xv) {
  int i = lut[zone_bin(z, v)];
  float xi = x[i];
  while (xi < v) { ++i; xi = x[i]; }
  LHCB_CHECK_IDX(i - z.b, z.e - z.b + 1);
  xv = xi;
  return i;
}
__device__ __forceinline__ int lower_bound(const float* __restrict__ x, const uint16_t* __restrict__ lut,
                                           const Zone& z, float v) {
  float xv;
  return lower_bound_v(x, lut, z, v, xv);
}
// first index in [b, e] with x[i] > v
__device__ __forceinline__ int upper_bound(const float* __restrict__ x, const uint16_t* __restrict__ lut,
                                           const Zone& z, float v) {
  v = fminf(v, 3.4028235e38f);                               // the +inf sentinel must end the scan
  int i = lut[zone_bin(z, v)];
  float xi = x[i];
  while (xi <= v) { ++i; xi = x[i]; }
  LHCB_CHECK_IDX(i - z.b, z.e - z.b + 1);
  return i;
}
// plain binary searches (global-memory arrays without a bin table)
__device__ __forceinline__ int lower_bound(const float* __restrict__ x, int b, int e, float v) {
  int n = e - b;
  while (n > 0) {
    const int h = n >> 1;
    const bool less = x[b + h] < v;
    b = less ? b + h + 1 : b;
    n = less ? n - h - 1 : h;
  }
  return b;
}
// largest t in [0, n) with offs[t] <= p (offs ascending, offs[0] = 0 <= p)
__device__ __forceinline__ int owner_of(const int* offs, int n, int p) {
  int b = 0;
  while (n > 1) {
    const int h = n >> 1;
    const bool le = offs[b + h] <= p;
    b = le ? b + h : b;
    n = le ? n - h : h;
  }
  return b;
}
// Index of the hit closest to xp with |x - xp| <= tol, ties to the lower index; -1 if none.  The zone is
// sorted, so with R the first hit >= xp and L = R - 1, every hit left of L is at least as far as L and every
// hit right of R at least as far as R (float subtraction is monotone): the minimum of |x - xp| is at L or R,
// "L if d_L <= d_R" keeps the lower index on a tie, and the only other hits with that same distance are equal
// neighbours further left (duplicates), which the walk back finds.  This is the hit the oracle's linear scan
// with "strictly closer replaces" selects.  The sentinels (-inf before, +inf after the zone) make every
// access safe and give the distance +inf.
__device__ __forceinline__ int closest_hit(const float* __restrict__ x, const uint16_t* __restrict__ lut,
                                           const Zone& z, float xp, float tol, float& xbest) {
  int i = lut[zone_bin(z, xp)];
  float xr = x[i];
  while (xr < xp) { ++i; xr = x[i]; }
  LHCB_CHECK_IDX(i - z.b, z.e - z.b + 1);
  const float xl = x[i - 1], xll = x[i - 2];                 // (i - 2 is at worst a sentinel or padding)
  const float dl = fabsf(xl - xp), dr = fabsf(xr - xp);
  const bool left = dl <= dr;
  const float d = left ? dl : dr;
  const bool ok = d <= tol;
  xbest = left ? xl : xr;
  i -= left;
  if (left && ok && fabsf(xll - xp) == d) {                 // duplicates: the lowest index among equal distances
    --i;
    while (fabsf(x[i - 1] - xp) == d) --i;
  }
  LHCB_CHECK_IDX(i - z.b, z.e - z.b + 1);
  return ok ? i : -1;
}

// exclusive prefix sum of one int per thread over the CTA; total returned to every thread.  `flip` selects
// one of the two warp_sums buffers and is toggled: a call may follow the previous one without a barrier.
template <int NT>
__device__ __forceinline__ int block_exscan(int v, int* warp_sums /* [2][kSeedThreadsMax / 32 + 1] */, int& flip, int& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int* ws = warp_sums + flip * (kSeedThreadsMax / 32 + 1);
  flip ^= 1;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) ws[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = lane < NT / 32 ? ws[lane] : 0;
#pragma unroll
    for (int o = 1; o < NT / 32; o <<= 1) {
      const int t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    if (lane < NT / 32) ws[lane] = w;                        // inclusive warp totals
  }
  __syncthreads();
  total = ws[NT / 32 - 1];
  const int base = warp ? ws[warp - 1] : 0;
  return base + inc - v;
}

__device__ __forceinline__ float xz_at(const SeedParams& p, float ax, float bx, float cx, int layer) {
  return (ax + bx * p.zb[layer]) + cx * p.gz[layer];       // Eq. 1
}

__device__ __forceinline__ unsigned long long clone_key(float chi2, float cx, int nx, int it) {
  float score = 1000.f * chi2;                              // Eq. 15, reading A8
  if (nx == 5) score = 10.f * score;
  return ((unsigned long long)__float_as_uint(score) << 32) |
         ((__float_as_uint(fabsf(cx)) & ~1u) | (unsigned)(it & 1));
}

// ------------------------------------------------------------------------------------ u/v walk
struct UvComb { int n, mask; float m[6]; int hit[6]; };
struct __align__(16) UvSuccess { uint16_t k; uint8_t pp, n; uint16_t hit[6]; };   // hit: tile index or 0xFFFF

// O9: theta = -Q[mask] m ; r = m + tan(alpha) (ay + by zb) ; chi2 = sum r^2 * wy[n]
__device__ __forceinline__ float fit_y(const SeedParams& p, const UvComb& c, float& ay, float& by) {
  const float* __restrict__ Q = p.Q + c.mask * 12;
  float th[2];
#pragma unroll
  for (int k = 0; k < 2; ++k) {
    float acc = 0.f;
    bool first = true;
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      if (!(c.mask >> s & 1)) continue;
      const float t = __ldg(Q + k * 6 + s) * c.m[s];
      acc = first ? t : acc + t;
      first = false;
    }
    th[k] = -acc;
  }
  float ssq = 0.f;
  bool first = true;
#pragma unroll
  for (int s = 0; s < 6; ++s) {
    if (!(c.mask >> s & 1)) continue;
    const int l = p.ul[s];
    const float rr = c.m[s] + p.tan_a[l] * (th[0] + th[1] * p.zb[l]);
    ssq = first ? rr * rr : ssq + rr * rr;
    first = false;
  }
  ay = th[0]; by = th[1];
  return ssq * p.wy[c.n];
}

// ------------------------------------------------------------------------------------ kernel
// one u/v walk that can still reach min_uv_hits after phase A: (owner << 16 | first hit), running t_y, the
// hits of the first three other stereo layers (tile index or 0xFFFF) and the hit count so far
struct __align__(16) UvLive { uint32_t item; float ty; uint16_t h[3]; uint16_t n; };

// O8, one layer of the walk: stereo slot s of the survivor whose predictions are xpk[0..5]; closest hit
// within tol of the prediction at the running t_y; a found hit updates t_y (A7) and the count.
__device__ __forceinline__ int uv_step(const SeedSmemHeader& H, const float* __restrict__ hx,
                                       const uint16_t* __restrict__ lut, const float* xpk, int s, float tol,
                                       float& ty, int& n) {
  const float4 cf = H.uvc[s];                                // {z tan(alpha), 1/tan(alpha), 1/z, layer}
  const int l = __float_as_int(cf.w);
  const float xs = xpk[s];
  const float xe = xs - ty * cf.x;
  const Zone z = H.zi[l];
  float xhh = 0.f;
  const int h = closest_hit(hx, lut + l * (kLutBins + 1), z, xe, tol, xhh);
  if (h >= 0) {
    const float yl = (xs - xhh) * cf.y;
    ty = 0.5f * (ty + yl * cf.z);
    ++n;
  }
  return h;
}

template <int NT, int MIN_CTAS>
__global__ void __launch_bounds__(NT, MIN_CTAS)
seeding_kernel(const __grid_constant__ SeedParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  SeedSmemHeader& H = *reinterpret_cast<SeedSmemHeader*>(smem);
  uint16_t* lut = reinterpret_cast<uint16_t*>(smem + kSeedHeaderBytes);
  uint16_t* kept = reinterpret_cast<uint16_t*>(smem + seed_off_kept());
  const int off_hits = (int)seed_off_hits(p.max_cand);
  float* hx = reinterpret_cast<float*>(smem + off_hits);
  Cand* cand_end = reinterpret_cast<Cand*>(smem + p.smem_total);               // candidate c lives at cand_end[-1 - c]

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  constexpr int T = NT, nwarps = NT / 32;
  const float inf = __int_as_float(0x7f800000);
  int flip = 0;                                            // buffer of the next block scan
  LHCB_CLK_INIT
  const int half_id = p.order ? (int)p.order[blockIdx.x] : (int)blockIdx.x, event = half_id >> 1, h = half_id & 1;
  const uint32_t* zo = p.zone_off + (size_t)half_id * 12;

  // ---- S0: stage the half's hits, every zone framed by sentinels ----------------------------------
  // The half is one contiguous run of hit_x: ONE bulk async copy brings its 16-byte aligned superset into a
  // staging buffer (the work region, empty so far); the zones are then moved into the tile, each as
  // [-inf, -inf, hits ..., +inf]: zone z starts at pos_z = 2 + sum_{k<z} (n_k + 3).
  uint32_t zoff[13];
#pragma unroll
  for (int z = 0; z < 13; ++z) zoff[z] = __ldg(zo + z);
  const int n_half = (int)(zoff[12] - zoff[0]);
  const uint32_t slot0 = (uint32_t)half_id * (uint32_t)p.max_seeds;
  bool zone_too_big = false;
#pragma unroll
  for (int z = 0; z < 12; ++z) zone_too_big |= zoff[z + 1] - zoff[z] >= (1u << kZoneIndexBits);
  if (n_half > p.max_hits || zone_too_big) {               // uniform: whole CTA leaves
    if (tid == 0) {
      p.count[half_id] = 0; p.status[half_id] = LHCB_ST_HITS_OVERFLOW;
      if (p.done) {                                          // published like every other exit: a dependent Matching CTA reads them
        __threadfence();
        asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p.done + half_id), "r"(1u) : "memory");
      }
    }
    return;
  }
  const int off_w = off_hits + (int)seed_tile_bytes(n_half);   // work region W: from the end of the tile to the first candidate slot
  float* stg = reinterpret_cast<float*>(smem + off_w);
  const uint32_t a0 = zoff[0] & ~3u;                       // 16-byte aligned start of the staged run
  uint32_t a1 = (zoff[12] + 3u) & ~3u;                     // end of the bulk part (multiple of 4 floats)
  if (a1 > (p.n_hits & ~3u)) a1 = p.n_hits & ~3u;
  if ((reinterpret_cast<uintptr_t>(p.hit_x) & 15) != 0 || a1 < a0) a1 = a0;
  const uint32_t mbar_addr = (uint32_t)__cvta_generic_to_shared(&H.mbar);
  if (tid == 0) {
    H.n_trip = 0; H.n_cand = 0; H.n_kept = 0; H.n_seed = 0; H.status = 0;
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_addr));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    const uint32_t bytes = (a1 - a0) * 4u;
    if (bytes > 0) {
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_addr), "r"(bytes) : "memory");
      asm volatile(
          "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
              (uint32_t)__cvta_generic_to_shared(stg)),
          "l"(p.hit_x + a0), "r"(bytes), "r"(mbar_addr)
          : "memory");
    } else {
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar_addr) : "memory");
    }
    int acc = 0, pos = 2, xs = 0;
#pragma unroll
    for (int z = 0; z < 12; ++z) {                         // x-hits are numbered densely for the clone table
      const int n = (int)(zoff[z + 1] - zoff[z]);
      if (xs < 6 && p.xl[xs] == z) { H.xoff[xs] = acc - pos; acc += n; ++xs; }
      pos += n + 3;
    }
    H.n_xhits = acc;
  }
  // tail (and the whole run when the source is not 16-byte aligned) with plain loads
  for (uint32_t i = (a1 > zoff[0] ? a1 : zoff[0]) + tid; i < zoff[12]; i += T) stg[i - a0] = __ldg(p.hit_x + i);
  if (tid >= 64 && tid < 70) {
    const int l = p.ul[tid - 64];
    H.uvc[tid - 64] = make_float4(p.zt[l], p.inv_tan[l], p.inv_z[l], __int_as_float(l));
  }
  {                                                        // bin tables: every entry "unmarked"
    uint32_t* L32 = reinterpret_cast<uint32_t*>(lut);
    constexpr int nw = (12 * (kLutBins + 1) + 1) / 2;
    for (int i = tid; i < nw; i += T) L32[i] = 0xFFFFFFFFu;
  }
  if (p.done && tid == 0) { p.done[half_id] = 0u; __threadfence(); }
  __syncthreads();                                         // the mbarrier is initialised; the tail hits are in place
  // programmatic dependent launch: once every CTA of this grid has passed this point (its flag is down), the
  // Matching grid may be scheduled into the SM resources the last wave leaves free; its CTAs wait on the flags
  if (p.done) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  {
    uint32_t done = 0;
    while (!done) {
      asm volatile(
          "{\n\t.reg .pred q;\n\t"
          "mbarrier.try_wait.parity.shared::cta.b64 q, [%1], 0;\n\t"
          "selp.u32 %0, 1, 0, q;\n\t}"
          : "=r"(done)
          : "r"(mbar_addr)
          : "memory");
    }
  }
  {
    int pos = 2;
#pragma unroll
    for (int z = 0; z < 12; ++z) {
      const int n = (int)(zoff[z + 1] - zoff[z]);
      const float* src = stg + (zoff[z] - a0);
      LHCB_CHECK_IDX(off_hits + (pos + n + 1) * 4, off_w + 1);
      for (int i = tid; i < n; i += T) hx[pos + i] = src[i];
      if (tid == 32 + z) {                                 // sentinels, bin function, index map of zone z
        hx[pos - 2] = -inf; hx[pos - 1] = -inf; hx[pos + n] = inf;
        float x0 = 0.f, invw = 0.f;
        if (n > 0) {
          x0 = src[0];
          const float span = src[n - 1] - x0;
          invw = span > 0.f ? (float)kLutBins / span : 0.f;
        }
        Zone zn; zn.b = pos; zn.e = pos + n; zn.x0 = x0; zn.invw = invw;
        H.zi[z] = zn;
        H.zg[z] = zoff[z] - (uint32_t)pos;
      }
      pos += n + 3;
    }
  }
  __syncthreads();
  LHCB_CLK(0)
  const int w_stat = p.smem_total - p.max_cand * (int)sizeof(Cand) - off_w;   // bytes of W with every candidate slot used
  Triplet* trip = reinterpret_cast<Triplet*>(smem + off_w);
  unsigned long long* tbl = reinterpret_cast<unsigned long long*>(smem + off_w);   // aliases trip
  const int trip_cap = w_stat / (int)sizeof(Triplet);
  // the first hit of every occupied bin marks its entry ...
#pragma unroll 1
  for (int z = 0; z < 12; ++z) {
    const Zone zz = H.zi[z];
    uint16_t* L = lut + z * (kLutBins + 1);
    for (int i = zz.b + tid; i < zz.e; i += T) {
      const int k1 = zone_bin(zz, hx[i]);
      const int k0 = zone_bin(zz, hx[i - 1]);              // -inf in front of the first hit: bin 0
      LHCB_CHECK_IDX(k1, kLutBins);
      if (i == zz.b || k1 != k0) L[k1] = (uint16_t)i;
    }
  }
  __syncthreads();
  // ... and every empty bin takes the entry of the next marked bin above it (zone end after the last one):
  // one warp per zone, 32 bins at a time from the top, the next marked bin of a lane from a ballot
  for (int z = warp; z < 12; z += nwarps) {
    uint16_t* L = lut + z * (kLutBins + 1);
    unsigned carry = (unsigned)H.zi[z].e;
    if (lane == 0) L[kLutBins] = (uint16_t)carry;
#pragma unroll 2
    for (int c = kLutBins / 32 - 1; c >= 0; --c) {
      const unsigned v = L[c * 32 + lane];
      const unsigned above = __ballot_sync(0xffffffffu, v != 0xFFFFu) >> lane;   // marked bins at or above mine
      const unsigned w = __shfl_sync(0xffffffffu, v, (lane + __ffs(above) - 1) & 31);
      const unsigned r = above ? w : carry;
      L[c * 32 + lane] = (uint16_t)r;
      carry = __shfl_sync(0xffffffffu, r, 0);
    }
  }
  __syncthreads();
  LHCB_CLK(1)

  // ---- S1 per iteration: two- and three-hit search, triplets of both iterations in one queue ----------
  // items of the pair walk live in the candidate slots (empty until S2): (i1 | first i3 << 13 | (n - 1) << 26)
  // one item buffer per iteration: the walk of iteration 0 needs no barrier before the T3 windows of iteration 1
  const int item_cap = p.max_cand * (int)(sizeof(Cand) / 8);
  for (int it = 0; it < 2; ++it) {
    uint32_t* items = reinterpret_cast<uint32_t*>(smem + p.smem_total - p.max_cand * (int)sizeof(Cand)) + it * item_cap;
    const int l1 = p.l1[it], l2 = p.l2[it], l3 = p.l3[it];
    const Zone z1n = H.zi[l1], z2n = H.zi[l2], z3n = H.zi[l3];
    const uint16_t* lut2 = lut + l2 * (kLutBins + 1);
    const uint16_t* lut3 = lut + l3 * (kLutBins + 1);
    const int b1 = z1n.b, n1 = z1n.e - z1n.b, b2 = z2n.b, b3 = z3n.b;
    const float r13 = p.r13[it], dx3 = p.dx3max[it], idz = p.inv_dz13[it], z1 = p.z1[it], dz12 = p.dz12[it];
    const float K = p.K[it];

    for (int tile0 = 0; tile0 < n1; tile0 += T) {
      // O2: T3 window of this thread's T1 hit, cut into items of at most kItemPairs T3 hits
      int cnt = 0, fst = 0;
      if (tile0 + tid < n1) {
        const float x1 = hx[b1 + tile0 + tid];
        const float c = x1 * r13;                                                // Eq. 11
        const float lo = c - dx3, hi = c + dx3;
        fst = lower_bound(hx, lut3, z3n, lo);
        cnt = upper_bound(hx, lut3, z3n, hi) - fst;
      }
      const int nit = (cnt + kItemPairs - 1) / kItemPairs;
      int total;
      const int ex = block_exscan<NT>(nit, &H.warp_sums[0][0], flip, total);
      if (total > item_cap) { total = item_cap; if (tid == 0) H.status |= LHCB_ST_TRIPLET_OVERFLOW; }
      {
        const uint32_t base = (uint32_t)(b1 + tile0 + tid) | ((uint32_t)fst << kTileIndexBits);
        int left = cnt;
        for (int q = 0; q < nit && ex + q < item_cap; ++q, left -= kItemPairs) {
          const int n = left < kItemPairs ? left : kItemPairs;
          items[ex + q] = base + ((uint32_t)(q * kItemPairs) << kTileIndexBits) + ((uint32_t)(n - 1) << (2 * kTileIndexBits));
        }
      }
      __syncthreads();
      LHCB_CLK(2)
      for (int i = tid; i < total; i += T) {
        const uint32_t item = items[i];
        const int i1 = (int)(item & ((1u << kTileIndexBits) - 1)), i3f = (int)((item >> kTileIndexBits) & ((1u << kTileIndexBits) - 1));
        const int n = (int)(item >> (2 * kTileIndexBits)) + 1;
        const float x1 = hx[i1];
        const int e2 = z2n.e;
        int j = e2;
        float xj = inf, lo2p = inf;
        for (int k = 0; k < n; ++k) {
          const float x3 = hx[i3f + k];
          const float t13 = (x3 - x1) * idz;                                     // O3, Eq. 4
          const float x0 = x1 - z1 * t13;                                        // Eq. 3
          const float invp = p.a * fabsf(x0) + p.b * (x0 * x0);                  // Eq. 5
          const float x2c = x1 + dz12 * t13;                                     // O4, Eq. 12
          const float kinv = p.kappa * invp;
          const float cxp = x0 >= 0.f ? -kinv : kinv;                            // A3
          const float ca = p.f_lo * cxp, cb = p.f_hi * cxp;                      // A4
          const float cxlo = fminf(ca, cb) - p.d_lo, cxhi = fmaxf(ca, cb) + p.d_hi;
          const float ea = x2c + K * cxlo, eb = x2c + K * cxhi;
          const float lo2 = fminf(ea, eb), hi2 = fmaxf(ea, eb);
          // the T2 interval moves up with x3: the pointer of the previous pair is a valid start; the first
          // pair of the item (and a lower edge that moved down, a rounding event) starts from the bin table
          if (lo2 < lo2p) { j = lut2[zone_bin(z2n, lo2)]; xj = hx[j]; }
          lo2p = lo2;
          while (xj < lo2) { ++j; xj = hx[j]; }
          LHCB_CHECK_IDX(j - b2, e2 - b2 + 1);
          int jj = j;
          float xjj = xj;
          while (xjj <= hi2) {
            if (jj >= e2) break;                                                 // hi2 = +inf: stop at the sentinel
            const int slot = smem_inc(&H.n_trip);
            LHCB_CHECK_IDX(jj - b2, e2 - b2);
            if (slot < trip_cap)
              trip[slot] = (uint32_t)(i1 - b1) | ((uint32_t)(jj - b2) << kZoneIndexBits) |
                           ((uint32_t)(i3f + k - b3) << (2 * kZoneIndexBits)) | ((uint32_t)it << (3 * kZoneIndexBits));
            ++jj;
            xjj = hx[jj];
          }
        }
      }
      if (it == 1 || tile0 + T < n1) __syncthreads();
      LHCB_CLK(3)
    }
  }
  __syncthreads();
  // ---- S2: extension of the queued triplets of both iterations (O5) ---------------------------------
  {
    int nt = H.n_trip;
    LHCB_DBG_MAX(0, nt)
    if (nt > trip_cap) { nt = trip_cap; if (tid == 0) H.status |= LHCB_ST_TRIPLET_OVERFLOW; }
    const int miss_max = 6 - p.min_x_hits;

    for (int t = tid; t < nt; t += T) {
      const Triplet tr = trip[t];
      const int it = (int)(tr >> (3 * kZoneIndexBits));      // the queue holds iteration 0 first: warps are uniform in it
      const int l1 = p.l1[it];
      constexpr uint32_t zmask = (1u << kZoneIndexBits) - 1;
      const int i1 = H.zi[l1].b + (int)(tr & zmask), i2 = H.zi[p.l2[it]].b + (int)((tr >> kZoneIndexBits) & zmask),
                i3 = H.zi[p.l3[it]].b + (int)((tr >> (2 * kZoneIndexBits)) & zmask);
      LHCB_CHECK_IDX(i1 - H.zi[l1].b, H.zi[l1].e - H.zi[l1].b); LHCB_CHECK_IDX(i2 - H.zi[p.l2[it]].b, H.zi[p.l2[it]].e - H.zi[p.l2[it]].b);
      LHCB_CHECK_IDX(i3 - H.zi[p.l3[it]].b, H.zi[p.l3[it]].e - H.zi[p.l3[it]].b);
      const float x1 = hx[i1], x2 = hx[i2], x3 = hx[i3];
      const float t13 = (x3 - x1) * p.inv_dz13[it];
      const float x2c = x1 + p.dz12[it] * t13;
      const float cx = (x2 - x2c) * p.inv_K[it];
      const float bx = t13 - cx * p.G13[it];
      const float ax = (x1 - bx * p.zb[l1]) - cx * p.gz[l1];
      int ho[3];
      int miss = 0, pattern = 0;
#pragma unroll
      for (int q = 0; q < 3; ++q) {                          // the three other x-layers in z order
        ho[q] = -1;
        if (miss > miss_max) continue;                        // too many layers missed already
        const int l = p.ol[it][q];
        const Zone z = H.zi[l];
        float xh;
        ho[q] = closest_hit(hx, lut + l * (kLutBins + 1), z, xz_at(p, ax, bx, cx, l), p.tol_x, xh);
        if (ho[q] < 0) { ++miss; pattern = 1 + p.os[it][q]; }
      }
      if (miss > miss_max) continue;
      // enough x-hits: queue the three-point parabola and its hits; the least-squares fit runs as a dense
      // pass over the queued candidates of both iterations (S2b)
      const int k = smem_inc(&H.n_cand);
      if (k < p.max_cand) {
        Cand& cd = cand_end[-1 - k];
        cd.ax = ax; cd.bx = bx; cd.cx = cx; cd.chi2 = 0.f;
        cd.hit[p.ss[it][0]] = (uint16_t)i1; cd.hit[p.ss[it][1]] = (uint16_t)i2; cd.hit[p.ss[it][2]] = (uint16_t)i3;
#pragma unroll
        for (int q = 0; q < 3; ++q) cd.hit[p.os[it][q]] = (uint16_t)ho[q];     // -1 -> 0xFFFF
        cd.nx = (uint8_t)(6 - miss); cd.it = (uint8_t)it; cd.keep = 0; cd.pattern = (uint8_t)pattern;
      }
    }
    __syncthreads();
    LHCB_CLK(4)
  }

  int nc = H.n_cand;
  LHCB_DBG_MAX(1, nc)
  if (nc > p.max_cand) { nc = p.max_cand; if (tid == 0) H.status |= LHCB_ST_CAND_OVERFLOW; }
  // ---- S2b: least-squares fit of every queued candidate (O6): fixed pseudo-inverse map per missing-layer
  // pattern applied to the residuals w.r.t. the three-point parabola
  for (int c = tid; c < nc; c += T) {
    Cand& cd = cand_end[-1 - c];
    const int pattern = cd.pattern;
    float ax = cd.ax, bx = cd.bx, cx = cd.cx;
    float r[6];
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      const int l = p.xl[s];
      r[s] = 0.f;
      if (pattern != 1 + s) r[s] = hx[cd.hit[s]] - xz_at(p, ax, bx, cx, l);
    }
    const float* __restrict__ P = p.P + pattern * 18;
    float d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      float acc = 0.f;
      bool first = true;
#pragma unroll
      for (int s = 0; s < 6; ++s) {
        if (pattern == 1 + s) continue;
        const float tt = __ldg(P + k * 6 + s) * r[s];
        acc = first ? tt : acc + tt;
        first = false;
      }
      d[k] = acc;
    }
    float ssq = 0.f;
    bool first = true;
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      if (pattern == 1 + s) continue;
      const int l = p.xl[s];
      const float rr = r[s] - ((d[0] + d[1] * p.zb[l]) + d[2] * p.gz[l]);
      ssq = first ? rr * rr : ssq + rr * rr;
      first = false;
    }
    const float chi2 = ssq * p.wx[cd.nx];
    cd.ax = ax + d[0]; cd.bx = bx + d[1]; cd.cx = cx + d[2]; cd.chi2 = chi2;
    if (chi2 > p.chi2x_max) cd.nx = 0;
  }
  __syncthreads();
  // ---- S3: clone kill (O7) ------------------------------------------------------------------
  const int n_xhits = H.n_xhits;
  if (n_xhits > (w_stat + (p.max_cand - nc) * (int)sizeof(Cand)) / 8) {   // uniform: the clone table does not fit
    if (tid == 0) {
      p.count[half_id] = 0; p.status[half_id] = H.status | LHCB_ST_HITS_OVERFLOW;
      if (p.done) { __threadfence(); p.done[half_id] = 1u; }
    }
    return;
  }
  for (int i = tid; i < n_xhits; i += T) tbl[i] = kNoKey;
  __syncthreads();
  for (int c = tid; c < nc; c += T) {
    const Cand& cd = cand_end[-1 - c];
    if (cd.nx == 0) continue;
    const unsigned long long key = clone_key(cd.chi2, cd.cx, cd.nx, cd.it);
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (cd.hit[s] != 0xFFFF) { LHCB_CHECK_IDX(H.xoff[s] + cd.hit[s], n_xhits); atomicMin(&tbl[H.xoff[s] + cd.hit[s]], key); }
  }
  __syncthreads();
  for (int c = tid; c < nc; c += T) {
    Cand& cd = cand_end[-1 - c];
    if (cd.nx == 0) continue;
    const unsigned long long key = clone_key(cd.chi2, cd.cx, cd.nx, cd.it);
    int own = 0;
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (cd.hit[s] != 0xFFFF && tbl[H.xoff[s] + cd.hit[s]] == key) ++own;
    const bool keep = own >= 3 || (own >= 2 && cd.nx == 6);
    cd.keep = keep;
    if (keep) { const int kk = smem_inc(&H.n_kept); LHCB_CHECK_IDX(kk, p.max_cand); kept[kk] = (uint16_t)c; }
  }
  __syncthreads();
  int nk = H.n_kept;
  LHCB_DBG_MAX(2, nk)
  // The clone table is dead.  The survivors move to the bottom of W; after that every candidate slot is
  // dead too and W extends to the end of shared memory:
  //   [survivors | best key per survivor | predictions per survivor | item chunk | live walks | success queue]
  // (Hough version: [... | votes | first hypothesis per survivor | selected clusters | success queue])
  const int wbytes = p.smem_total - off_w;
  {                                                            // survivors must fit below the candidate slots (the
    // copy is in place) and leave room for the queues: 72 bytes per survivor, 132 with the Hough tables
    int nk_max = (wbytes - 4096) / (p.uv_hough ? 136 : 72);
    if (nk_max > w_stat / 32) nk_max = w_stat / 32;
    if (nk > nk_max) { nk = nk_max > 0 ? nk_max : 0; if (tid == 0) H.status |= LHCB_ST_UV_QUEUE_OVERFLOW; }
  }
  Cand* surv = reinterpret_cast<Cand*>(smem + off_w);
  LHCB_CHECK_IDX(nk * 72, wbytes + 1);
  for (int k = tid; k < nk; k += T) { LHCB_CHECK_IDX((int)kept[k], nc); surv[k] = cand_end[-1 - (int)kept[k]]; }
  unsigned long long* best = reinterpret_cast<unsigned long long*>(surv + nk);
  float* xps = reinterpret_cast<float*>(best + ((nk + 1) & ~1));          // [nk][8], 16-byte aligned: x_pred per stereo layer
  const int rest = wbytes - nk * 32 - ((nk + 1) & ~1) * 8 - nk * 32;      // >= 4096 - 8
  int C = (rest / 2) / 20;                                                // items per chunk: 4 B item + 16 B live walk
  C = C >= T ? C / T * T : (C & ~31);                                     // whole rounds of the CTA when possible
  if (C < 32) C = 32;
  uint32_t* uitems = reinterpret_cast<uint32_t*>(xps + (size_t)nk * 8);
  UvLive* live = reinterpret_cast<UvLive*>(uitems + C);
  UvSuccess* succ = reinterpret_cast<UvSuccess*>(live + C);
  int succ_cap = (rest - C * 20) / (int)sizeof(UvSuccess);
  __syncthreads();
  for (int k = tid; k < nk; k += T) {
    best[k] = kNoKey;
    const Cand& cd = surv[k];
#pragma unroll
    for (int s = 0; s < 6; ++s) xps[k * 8 + s] = xz_at(p, cd.ax, cd.bx, cd.cx, p.ul[s]);
  }
  if (tid == 0) H.n_trip = 0;                                            // reused as the success counter
  __syncthreads();
  LHCB_CLK(5)

  // ---- S4: u/v addition (O8, O9) --------------------------------------------------------------
  // owners w = 2*k + pass (k-th survivor); items = first-layer hits in the window of Eq. 16.  Every item
  // is queued as (owner, hit); phase A walks the first three other stereo layers of every item (dense),
  // the walks that can still reach min_uv_hits are queued with their state; phase B finishes them.
  const int sf0 = p.slot_of_layer[p.uv_first[0]], sf1 = p.slot_of_layer[p.uv_first[1]];
  if (p.uv_hough) {
    // ---- S4h: Hough-cluster version (O8h).  The queue space after the predictions is laid out as
    //   [votes u64[nk][6] | first hypothesis of each survivor int[nk + 1] | selected clusters u8[nk][8] | success queue]
    unsigned long long* vote = reinterpret_cast<unsigned long long*>(uitems);     // 16-byte aligned
    int* hoff = reinterpret_cast<int*>(vote + (size_t)nk * 6);
    uint8_t* selb = reinterpret_cast<uint8_t*>(hoff + nk + 1);
    const int hused = nk * 48 + (int)((((size_t)nk + 1) * 4 + (size_t)nk * 8 + 15) & ~(size_t)15);
    UvSuccess* hsucc = reinterpret_cast<UvSuccess*>(reinterpret_cast<unsigned char*>(uitems) + hused);
    const int hsucc_cap = (rest - hused) / (int)sizeof(UvSuccess);        // > 0: nk was clamped with the Hough tables in mind
    // H1: votes.  Owner = (survivor, stereo slot); every hit in the slot's window of Eq. 16 sets the bit of
    // its t_y bin (a layer counts once per bin)
    for (int w = tid; w < 6 * nk; w += T) {
      const int k = w / 6, sl = w - 6 * k;
      const float4 cf = H.uvc[sl];                                                // {z tan, 1/tan, 1/z, layer}
      const int l = __float_as_int(cf.w);
      const float xpl = xps[k * 8 + sl];
      const float wa = xpl - p.ywin_a[h][l], wb = xpl - p.ywin_b[h][l];
      const Zone zf = H.zi[l];
      const uint16_t* lutf = lut + l * (kLutBins + 1);
      float xh;
      int i = lower_bound_v(hx, lutf, zf, fminf(wa, wb), xh);
      const float whi = fminf(fmaxf(wa, wb), 3.4028235e38f);
      unsigned long long m = 0ull;
      while (xh <= whi) {
        const float t = ((xpl - xh) * cf.y) * cf.z;                               // Eq. 16, A7
        float tb = (t - p.h_tlo[h]) * p.h_invw;
        tb = fminf(fmaxf(tb, 0.f), 63.f);
        m |= 1ull << (int)tb;
        ++i;
        xh = hx[i];
      }
      vote[w] = m;
    }
    __syncthreads();
    // H2: cluster = bin + upper neighbour; population = layers voting in it, counted for all 64 bins at once
    // with a bit-sliced adder; up to eight clusters, most populated first, then lower t_y.  A block scan
    // gives every survivor the index of its first hypothesis (4 per cluster).
    int nhyp = 0;
    for (int tile0 = 0; tile0 < nk; tile0 += T) {
      const int k = tile0 + tid;
      int nsel = 0;
      if (k < nk) {
        unsigned long long ones = 0ull, twos = 0ull, fours = 0ull;
#pragma unroll
        for (int sl = 0; sl < 6; ++sl) {
          const unsigned long long m = vote[k * 6 + sl];
          const unsigned long long cm = m | (m >> 1);
          const unsigned long long c1 = ones & cm;
          ones ^= cm;
          const unsigned long long c2 = twos & c1;
          twos ^= c1;
          fours |= c2;
        }
        for (int level = 6; level >= p.min_uv_hits && level >= 1 && nsel < 8; --level) {
          unsigned long long lm = ((level & 4) ? fours : ~fours) & ((level & 2) ? twos : ~twos) & ((level & 1) ? ones : ~ones);
          while (lm && nsel < 8) {
            selb[k * 8 + nsel++] = (uint8_t)(__ffsll((long long)lm) - 1);
            lm &= lm - 1;
          }
        }
      }
      int total;
      const int ex = block_exscan<NT>(4 * nsel, &H.warp_sums[0][0], flip, total);
      if (k < nk) hoff[k] = nhyp + ex;
      nhyp += total;
    }
    if (tid == 0) hoff[nk] = nhyp;
    __syncthreads();
    // H3: thread per hypothesis: closest hit within tol_uv of the fixed line in every stereo layer
    for (int i = tid; i < nhyp; i += T) {
      const int k = owner_of(hoff, nk, i), j = i - hoff[k];                       // j = cluster rank * 4 + finer index
      const float* xpk = xps + k * 8;
      const float f = (float)(j & 3) * 0.5f + 0.25f;
      const float ty = p.h_tlo[h] + ((float)selb[k * 8 + (j >> 2)] + f) * p.h_w;
      int n = 0, hh[6];
#pragma unroll
      for (int sl = 0; sl < 6; ++sl) {
        hh[sl] = -1;
        if (n + (6 - sl) < p.min_uv_hits) continue;                               // cannot reach min_uv_hits any more
        const float4 cf = H.uvc[sl];
        const int l = __float_as_int(cf.w);
        const Zone z = H.zi[l];
        float xhh;
        hh[sl] = closest_hit(hx, lut + l * (kLutBins + 1), z, xpk[sl] - ty * cf.x, p.tol_uv, xhh);
        n += hh[sl] >= 0;
      }
      if (n < p.min_uv_hits) continue;
      const int slot = smem_inc(&H.n_trip);
      if (slot < hsucc_cap) {
        UvSuccess& u = hsucc[slot];
        u.k = (uint16_t)k; u.pp = (uint8_t)j; u.n = (uint8_t)n;
#pragma unroll
        for (int sl = 0; sl < 6; ++sl) u.hit[sl] = (uint16_t)hh[sl];
      }
    }
    __syncthreads();
    succ = hsucc;
    succ_cap = hsucc_cap;
  } else
  for (int tile0 = 0; tile0 < 2 * nk; tile0 += T) {
    const int nown = 2 * nk - tile0 < T ? 2 * nk - tile0 : T;
    int cnt = 0, fst = 0;
    if (tid < nown) {
      const int w = tile0 + tid, pp = w & 1;
      const int lf = p.uv_first[pp];
      const float xpf = xps[(w >> 1) * 8 + (pp ? sf1 : sf0)];
      const float wa = xpf - p.ywin_a[h][lf], wb = xpf - p.ywin_b[h][lf];
      const float wlo = wa < wb ? wa : wb, whi = wa > wb ? wa : wb;
      const Zone zf = H.zi[lf];
      const uint16_t* lutf = lut + lf * (kLutBins + 1);
      fst = lower_bound(hx, lutf, zf, wlo);
      cnt = upper_bound(hx, lutf, zf, whi) - fst;
    }
    int total;
    const int ex = block_exscan<NT>(cnt, &H.warp_sums[0][0], flip, total);
    LHCB_CLK(6)
    for (int q0 = 0; q0 < total; q0 += C) {                  // uniform: chunks of C items
      if (tid == 0) H.n_live = 0;
      {
        int i = q0 - ex; if (i < 0) i = 0;
        int iend = q0 + C - ex; if (iend > cnt) iend = cnt;
        for (; i < iend; ++i) { LHCB_CHECK_IDX(ex + i - q0, C); uitems[ex + i - q0] = ((uint32_t)tid << 16) | (uint32_t)(fst + i); }
      }
      __syncthreads();
      const int nitems = total - q0 < C ? total - q0 : C;
      for (int i = tid; i < nitems; i += T) {                // phase A
        const uint32_t item = uitems[i];
        const int w = tile0 + (int)(item >> 16), ih = (int)(item & 0xFFFFu);
        const int sf = (w & 1) ? sf1 : sf0;
        const float* xpk = xps + (w >> 1) * 8;
        const float4 cf = H.uvc[sf];
        const float y0 = (xpk[sf] - hx[ih]) * cf.y;          // Eq. 16
        float ty = y0 * cf.z;
        int n = 1;
        const int h0 = uv_step(H, hx, lut, xpk, 0 + (0 >= sf), p.tol_uv, ty, n);
        const int h1 = uv_step(H, hx, lut, xpk, 1 + (1 >= sf), p.tol_uv, ty, n);
        const int h2 = uv_step(H, hx, lut, xpk, 2 + (2 >= sf), p.tol_uv, ty, n);
        if (n + 2 < p.min_uv_hits) continue;                 // cannot reach min_uv_hits any more
        UvLive lv;
        lv.item = ((uint32_t)w << 16) | (uint32_t)ih; lv.ty = ty;
        lv.h[0] = (uint16_t)h0; lv.h[1] = (uint16_t)h1; lv.h[2] = (uint16_t)h2; lv.n = (uint16_t)n;
        const int ls = smem_inc(&H.n_live);
        LHCB_CHECK_IDX(ls, C);
        live[ls] = lv;
      }
      __syncthreads();
      const int nl = H.n_live;
      for (int i = tid; i < nl; i += T) {                    // phase B
        const UvLive lv = live[i];
        const int w = (int)(lv.item >> 16), ih = (int)(lv.item & 0xFFFFu);
        const int sf = (w & 1) ? sf1 : sf0;
        const float* xpk = xps + (w >> 1) * 8;
        float ty = lv.ty;
        int n = lv.n;
        const int h3 = uv_step(H, hx, lut, xpk, 3 + (3 >= sf), p.tol_uv, ty, n);
        const int h4 = (n + 1 < p.min_uv_hits) ? -1 : uv_step(H, hx, lut, xpk, 4 + (4 >= sf), p.tol_uv, ty, n);
        if (n < p.min_uv_hits) continue;
        const int slot = smem_inc(&H.n_trip);            // enough hits: queue for the dense fit pass
        if (slot < succ_cap) {
          UvSuccess& u = succ[slot];
          u.k = (uint16_t)(w >> 1); u.pp = (uint8_t)(w & 1); u.n = (uint8_t)n;
          u.hit[sf] = (uint16_t)ih;
          u.hit[0 + (0 >= sf)] = lv.h[0]; u.hit[1 + (1 >= sf)] = lv.h[1]; u.hit[2 + (2 >= sf)] = lv.h[2];
          u.hit[3 + (3 >= sf)] = (uint16_t)h3; u.hit[4 + (4 >= sf)] = (uint16_t)h4;
        }
      }
      __syncthreads();
    }
    LHCB_CLK(7)
  }
  int nsucc = H.n_trip;
  LHCB_DBG_MAX(3, nsucc)
  if (nsucc > succ_cap) { nsucc = succ_cap; if (tid == 0) H.status |= LHCB_ST_UV_QUEUE_OVERFLOW; }

  // ---- S5: y fit of every queued combination, best per survivor, seeds (O9, O10) ------------------
  const int pol = p.pol ? (int)p.pol[event] : p.polarity;
  const bool single = nsucc <= T;                              // the usual case: one combination per thread
  UvSuccess u;
  float ay = 0.f, by = 0.f, chi2y = 0.f;
  unsigned long long key = kNoKey;
  auto fit_success = [&](int i) {
    u = succ[i];
    UvComb c;
    c.n = u.n; c.mask = 0;
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      c.m[s] = 0.f; c.hit[s] = -1;
      if (u.hit[s] != 0xFFFF) { c.m[s] = hx[u.hit[s]] - xps[u.k * 8 + s]; c.mask |= 1 << s; }
    }
    chi2y = fit_y(p, c, ay, by);
    key = kNoKey;
    if (!(chi2y > p.chi2y_max)) {
      // ties: earlier pass, then lower first hit (iterative); earlier (cluster, finer index) (Hough)
      unsigned long long tie = u.pp;
      if (!p.uv_hough) {
        const int sf = p.slot_of_layer[p.uv_first[u.pp]];
        int first_local = 0;
#pragma unroll
        for (int s = 0; s < 6; ++s) first_local = (s == sf) ? (int)u.hit[s] - H.zi[p.ul[s]].b : first_local;
        tie = ((unsigned long long)u.pp << 16) | (unsigned long long)first_local;
      }
      key = ((unsigned long long)(6 - u.n) << 49) | ((unsigned long long)__float_as_uint(chi2y) << 17) | tie;
    }
  };
  for (int i = tid; i < nsucc; i += T) {
    fit_success(i);
    LHCB_CHECK_IDX(u.k, nk);
    if (key != kNoKey) atomicMin(&best[u.k], key);
  }
  __syncthreads();
  for (int i = tid; i < nsucc; i += T) {
    if (!single) fit_success(i);                               // more than one round: redo the (cheap) fit
    if (key == kNoKey || best[u.k] != key) continue;           // not the best combination of its survivor
    const Cand& cd = surv[u.k];
    const int slot = smem_inc(&H.n_seed);
    if (slot >= p.max_seeds) continue;
    const size_t o = (size_t)slot0 + slot, ct = p.cap_total;
    p.state[0 * ct + o] = (cd.ax + cd.bx * p.zbS) + cd.cx * p.gS;
    p.state[1 * ct + o] = ay + by * p.zbS;
    p.state[2 * ct + o] = cd.bx + cd.cx * p.gpS;
    p.state[3 * ct + o] = by;
    const float q = cd.cx * p.inv_kappa;
    p.state[4 * ct + o] = pol > 0 ? q : -q;
    p.par[0 * ct + o] = cd.ax; p.par[1 * ct + o] = cd.bx; p.par[2 * ct + o] = cd.cx;
    p.par[3 * ct + o] = ay; p.par[4 * ct + o] = by; p.par[5 * ct + o] = cd.chi2; p.par[6 * ct + o] = chi2y;
#pragma unroll
    for (int s = 0; s < 6; ++s) {
      const int lx = p.xl[s], lu = p.ul[s];
      p.hits[(size_t)lx * ct + o] = cd.hit[s] == 0xFFFF ? LHCB_NO_HIT : H.zg[lx] + (uint32_t)cd.hit[s];
      p.hits[(size_t)lu * ct + o] = u.hit[s] == 0xFFFF ? LHCB_NO_HIT : H.zg[lu] + (uint32_t)u.hit[s];
    }
    p.nx[o] = cd.nx;
    p.nuv[o] = u.n;
  }
  __syncthreads();
  LHCB_CLK(8)
  if (tid == 0) {
    int ns = H.n_seed;
    unsigned st = H.status;
    if (ns > p.max_seeds) { ns = p.max_seeds; st |= LHCB_ST_SEED_OVERFLOW; }
    p.count[half_id] = (uint32_t)ns;
    p.status[half_id] = st;
    if (p.done) {                                            // every seed store of the CTA precedes the barrier above
      __threadfence();
      asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p.done + half_id), "r"(1u) : "memory");
    }
  }
}

}  // namespace lhcb
