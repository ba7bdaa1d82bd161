// SciFi Seeding kernel (section 3) for sm_100a.
//
// One CTA per event-half (L372): the half's twelve sorted hit zones are staged into shared memory
// with one bulk async copy (cp.async.bulk + mbarrier) and stay there for every step (L370).
// Stages, separated by __syncthreads():
//   S1  two-hit + three-hit search     warp per T1 hit, lanes over the T3 window (Eq. 8-11),
//                                      per pair Eq. 3-5 and the T2 band (Eq. 12-13, A3/A4);
//                                      triplets are queued in shared memory
//   S2  extension + fit                thread per queued triplet: exact parabola, +-1 mm closest hit in
//                                      the other three x-layers, >=5 hits, fixed-matrix least squares (L90)
//   S3  clone kill                     64-bit atomicMin table per x-hit, vote pass (L183-200, Eq. 15)
//   S4  u/v addition                   8-lane group per (survivor, pass), lanes over first-layer hits
//                                      (Eq. 16); best combination by packed-key min
//   S5  seed output                    thread per survivor: rebuild the winning combination, y fit, store
//
// Arithmetic: every formula follows DESIGN.md "Arithmetic specification" operation by operation;
// this translation unit is compiled with -fmad=false so that no multiply-add is contracted.
#pragma once
#include <cstdint>

#include "../../include/lhcb.h"

namespace lhcb {

constexpr int kSeedThreads = 256;
constexpr int kUvGroup = 8;
constexpr unsigned long long kNoKey = ~0ull;

struct SeedParams {
  float zb[12], gz[12], tan_a[12], inv_tan[12], inv_z[12], zt[12];
  float ywin_a[2][12], ywin_b[2][12];
  int xl[6], ul[6], slot_of_layer[12];
  int l1[2], l2[2], l3[2];
  float dx3max[2], r13[2], inv_dz13[2], z1[2], dz12[2], K[2], inv_K[2], G13[2];
  float a, b, kappa, inv_kappa, f_lo, f_hi, d_lo, d_hi, tol_x, tol_uv, chi2x_max, chi2y_max;
  float wx[7], wy[7];
  float zbS, gS, gpS;
  int min_x_hits, min_uv_hits, uv_first[2], polarity;
  int max_seeds, max_cand, max_hits, max_trip;
  const float* P;   // [7][3][6]
  const float* Q;   // [64][2][6]
  // batch
  int n_events;
  uint32_t n_hits;
  const uint32_t* zone_off;
  const float* hit_x;
  const int8_t* pol;
  uint32_t* count;
  float* state;
  float* par;
  uint32_t* hits;
  uint8_t* nx;
  uint8_t* nuv;
  uint32_t* status;
  size_t cap_total;
};

struct __align__(8) Triplet { uint16_t i1, i2, i3, it; };                 // zone-local indices
struct __align__(16) Cand { float ax, bx, cx, chi2; uint16_t hit[6]; uint8_t nx, it, keep, pad; };

struct SeedSmemHeader {
  unsigned long long mbar;
  int zl[13];          // zone offsets relative to the staged tile
  int xbase[7];        // prefix of x-zone sizes (clone-table index base per x-slot)
  int n_trip, n_cand, n_kept, n_seed;
  unsigned int status;
};

__host__ __device__ inline size_t seed_smem_bytes(int max_hits, int max_cand, int max_trip) {
  size_t b = 256;                                          // header
  b += ((size_t)max_hits + 8) * 4;                         // hits tile (16-byte aligned superset)
  b = (b + 15) & ~(size_t)15;
  b += (size_t)max_cand * sizeof(Cand);
  b += (size_t)max_cand * 2;                               // kept list
  b = (b + 15) & ~(size_t)15;
  b += (size_t)max_trip * 8;                               // triplet queue / clone table / best keys
  return b;
}

// ------------------------------------------------------------------------------------ searches
// first index in [b, e) with x[i] >= v
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
// first index in [b, e) with x[i] > v
__device__ __forceinline__ int upper_bound(const float* __restrict__ x, int b, int e, float v) {
  int n = e - b;
  while (n > 0) {
    const int h = n >> 1;
    const bool le = x[b + h] <= v;
    b = le ? b + h + 1 : b;
    n = le ? n - h - 1 : h;
  }
  return b;
}
// index of the hit closest to xp with |x - xp| <= tol, ties to the lower index; -1 if none
__device__ __forceinline__ int closest_hit(const float* __restrict__ x, int b, int e, float xp, float tol) {
  const int j = lower_bound(x, b, e, xp);
  int best = -1;
  float bd = 0.f;
  if (j > b) {
    int l = j - 1;
    const float xl = x[l];
    while (l > b && x[l - 1] == xl) --l;     // equal x: the lower index wins
    const float d = fabsf(xl - xp);
    if (d <= tol) { best = l; bd = d; }
  }
  if (j < e) {
    const float d = fabsf(x[j] - xp);
    if (d <= tol && (best < 0 || d < bd)) best = j;
  }
  return best;
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

// O8 for one first-layer hit ih (tile index) of pass pp: closest hits within tol_uv in the other
// five stereo layers, running-average t_y (A7).
__device__ __forceinline__ void uv_walk(const SeedParams& p, const float* __restrict__ hx, const int* zl,
                                        const float* xp, int sf, int ih, UvComb& c) {
  const int lf = p.ul[sf];
  const float xh = hx[ih];
  const float y0 = (xp[sf] - xh) * p.inv_tan[lf];          // Eq. 16
  float ty = y0 * p.inv_z[lf];
#pragma unroll
  for (int s = 0; s < 6; ++s) { c.hit[s] = -1; c.m[s] = 0.f; }
  c.hit[sf] = ih; c.m[sf] = xh - xp[sf]; c.mask = 1 << sf; c.n = 1;
#pragma unroll
  for (int s = 0; s < 6; ++s) {
    if (s == sf) continue;
    const int l = p.ul[s];
    const float xe = xp[s] - ty * p.zt[l];
    const int h = closest_hit(hx, zl[l], zl[l + 1], xe, p.tol_uv);
    if (h >= 0) {
      const float xhh = hx[h];
      const float yl = (xp[s] - xhh) * p.inv_tan[l];
      ty = 0.5f * (ty + yl * p.inv_z[l]);
      c.hit[s] = h; c.m[s] = xhh - xp[s]; c.mask |= 1 << s; ++c.n;
    }
  }
}

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
__global__ void __launch_bounds__(kSeedThreads)
seeding_kernel(const __grid_constant__ SeedParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  SeedSmemHeader& H = *reinterpret_cast<SeedSmemHeader*>(smem);
  float* hx = reinterpret_cast<float*>(smem + 256);
  size_t off = 256 + ((size_t)p.max_hits + 8) * 4;
  off = (off + 15) & ~(size_t)15;
  Cand* cand = reinterpret_cast<Cand*>(smem + off);
  off += (size_t)p.max_cand * sizeof(Cand);
  uint16_t* kept = reinterpret_cast<uint16_t*>(smem + off);
  off += (size_t)p.max_cand * 2;
  off = (off + 15) & ~(size_t)15;
  Triplet* trip = reinterpret_cast<Triplet*>(smem + off);
  unsigned long long* tbl = reinterpret_cast<unsigned long long*>(smem + off);   // aliases trip

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nwarps = kSeedThreads / 32;
  const int half_id = blockIdx.x, event = half_id >> 1, h = half_id & 1;
  const uint32_t* zo = p.zone_off + (size_t)half_id * 12;

  const uint32_t g_begin = zo[0], g_end = zo[12];
  const uint32_t a0 = g_begin & ~3u;                       // 16-byte aligned start of the staged tile
  const int n_half = (int)(g_end - g_begin);
  const uint32_t slot0 = (uint32_t)half_id * (uint32_t)p.max_seeds;

  if (n_half > p.max_hits) {                               // uniform: whole CTA leaves
    if (tid == 0) { p.count[half_id] = 0; p.status[half_id] = LHCB_ST_HITS_OVERFLOW; }
    return;
  }

  // ---- S0: stage the half's hits -----------------------------------------------------
  const bool aligned = ((reinterpret_cast<uintptr_t>(p.hit_x) & 15) == 0);
  uint32_t a1 = (g_end + 3u) & ~3u;                        // end of the bulk part (multiple of 4 floats)
  if (a1 > (p.n_hits & ~3u)) a1 = p.n_hits & ~3u;
  if (!aligned || a1 < a0) a1 = a0;
  const uint32_t mbar_addr = (uint32_t)__cvta_generic_to_shared(&H.mbar);
  if (tid == 0) {
    H.n_trip = 0; H.n_cand = 0; H.n_kept = 0; H.n_seed = 0; H.status = 0;
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_addr));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (tid < 13) H.zl[tid] = (int)(zo[tid] - a0);
  __syncthreads();
  if (tid == 0) {
    int acc = 0;
    for (int s = 0; s < 6; ++s) { H.xbase[s] = acc; acc += H.zl[p.xl[s] + 1] - H.zl[p.xl[s]]; }
    H.xbase[6] = acc;
    const uint32_t bytes = (a1 - a0) * 4u;
    if (bytes > 0) {
      asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_addr), "r"(bytes) : "memory");
      asm volatile(
          "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
              (uint32_t)__cvta_generic_to_shared(hx)),
          "l"(p.hit_x + a0), "r"(bytes), "r"(mbar_addr)
          : "memory");
    } else {
      asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar_addr) : "memory");
    }
  }
  // tail (and the whole tile when the source is not 16-byte aligned) with plain loads
  for (uint32_t i = a1 + tid; i < g_end; i += kSeedThreads) hx[i - a0] = p.hit_x[i];
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
  __syncthreads();
  const int* zl = H.zl;
  if (H.xbase[6] > p.max_trip) {                            // clone table would not fit
    if (tid == 0) { p.count[half_id] = 0; p.status[half_id] = LHCB_ST_HITS_OVERFLOW; }
    return;
  }

  // ---- S1 + S2 per iteration -----------------------------------------------------------
  for (int it = 0; it < 2; ++it) {
    const int l1 = p.l1[it], l2 = p.l2[it], l3 = p.l3[it];
    const int b1 = zl[l1], e1 = zl[l1 + 1], b2 = zl[l2], e2 = zl[l2 + 1], b3 = zl[l3], e3 = zl[l3 + 1];
    const float r13 = p.r13[it], dx3 = p.dx3max[it], idz = p.inv_dz13[it], z1 = p.z1[it], dz12 = p.dz12[it];
    const float K = p.K[it];

    for (int i1 = b1 + warp; i1 < e1; i1 += nwarps) {                          // O2
      const float x1 = hx[i1];
      const float c = x1 * r13;                                                // Eq. 11
      const float lo = c - dx3, hi = c + dx3;
      const int first = lower_bound(hx, b3, e3, lo), last = upper_bound(hx, b3, e3, hi);
      for (int i3 = first + lane; i3 < last; i3 += 32) {
        const float x3 = hx[i3];
        const float t13 = (x3 - x1) * idz;                                     // O3, Eq. 4
        const float x0 = x1 - z1 * t13;                                        // Eq. 3
        const float invp = p.a * fabsf(x0) + p.b * (x0 * x0);                  // Eq. 5
        const float x2c = x1 + dz12 * t13;                                     // O4, Eq. 12
        const float kinv = p.kappa * invp;
        const float cxp = x0 >= 0.f ? -kinv : kinv;                            // A3
        const float ca = p.f_lo * cxp, cb = p.f_hi * cxp;                      // A4
        const float cxlo = (ca < cb ? ca : cb) - p.d_lo, cxhi = (ca > cb ? ca : cb) + p.d_hi;
        const float ea = x2c + K * cxlo, eb = x2c + K * cxhi;
        const float lo2 = ea < eb ? ea : eb, hi2 = ea > eb ? ea : eb;
        int j = lower_bound(hx, b2, e2, lo2);
        while (j < e2 && hx[j] <= hi2) {
          const int k = atomicAdd(&H.n_trip, 1);
          if (k < p.max_trip) {
            Triplet t;
            t.i1 = (uint16_t)(i1 - b1); t.i2 = (uint16_t)(j - b2); t.i3 = (uint16_t)(i3 - b3); t.it = (uint16_t)it;
            trip[k] = t;
          }
          ++j;
        }
      }
    }
    __syncthreads();
    int nt = H.n_trip;
    if (nt > p.max_trip) { nt = p.max_trip; if (tid == 0) H.status |= LHCB_ST_TRIPLET_OVERFLOW; }

    for (int t = tid; t < nt; t += kSeedThreads) {                             // O5 + O6
      const Triplet tr = trip[t];
      const int i1 = b1 + tr.i1, i2 = b2 + tr.i2, i3 = b3 + tr.i3;
      const float x1 = hx[i1], x2 = hx[i2], x3 = hx[i3];
      const float t13 = (x3 - x1) * idz;
      const float x2c = x1 + dz12 * t13;
      float cx = (x2 - x2c) * p.inv_K[it];
      float bx = t13 - cx * p.G13[it];
      float ax = (x1 - bx * p.zb[l1]) - cx * p.gz[l1];
      float r[6];
      int hit[6];
      int nx = 0, pattern = 0;
#pragma unroll
      for (int s = 0; s < 6; ++s) {
        const int l = p.xl[s];
        const float xp = xz_at(p, ax, bx, cx, l);
        int hh;
        if (l == l1) hh = i1;
        else if (l == l2) hh = i2;
        else if (l == l3) hh = i3;
        else hh = closest_hit(hx, zl[l], zl[l + 1], xp, p.tol_x);
        if (hh < 0) { hit[s] = -1; pattern = 1 + s; r[s] = 0.f; }
        else { hit[s] = hh - zl[l]; r[s] = hx[hh] - xp; ++nx; }
      }
      if (nx < p.min_x_hits) continue;
      // fixed-matrix least squares on the residuals w.r.t. the three-point parabola
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
      ax = ax + d[0]; bx = bx + d[1]; cx = cx + d[2];
      const float chi2 = ssq * p.wx[nx];
      if (chi2 > p.chi2x_max) continue;
      const int k = atomicAdd(&H.n_cand, 1);
      if (k < p.max_cand) {
        Cand cd;
        cd.ax = ax; cd.bx = bx; cd.cx = cx; cd.chi2 = chi2;
#pragma unroll
        for (int s = 0; s < 6; ++s) cd.hit[s] = hit[s] < 0 ? (uint16_t)0xFFFF : (uint16_t)hit[s];
        cd.nx = (uint8_t)nx; cd.it = (uint8_t)it; cd.keep = 0; cd.pad = 0;
        cand[k] = cd;
      }
    }
    __syncthreads();
    if (tid == 0) H.n_trip = 0;
    __syncthreads();
  }

  // ---- S3: clone kill (O7) ------------------------------------------------------------------
  int nc = H.n_cand;
  if (nc > p.max_cand) { nc = p.max_cand; if (tid == 0) H.status |= LHCB_ST_CAND_OVERFLOW; }
  const int n_xhits = H.xbase[6];
  for (int i = tid; i < n_xhits; i += kSeedThreads) tbl[i] = kNoKey;
  __syncthreads();
  for (int c = tid; c < nc; c += kSeedThreads) {
    const Cand& cd = cand[c];
    const unsigned long long key = clone_key(cd.chi2, cd.cx, cd.nx, cd.it);
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (cd.hit[s] != 0xFFFF) atomicMin(&tbl[H.xbase[s] + cd.hit[s]], key);
  }
  __syncthreads();
  for (int c = tid; c < nc; c += kSeedThreads) {
    Cand& cd = cand[c];
    const unsigned long long key = clone_key(cd.chi2, cd.cx, cd.nx, cd.it);
    int own = 0;
#pragma unroll
    for (int s = 0; s < 6; ++s)
      if (cd.hit[s] != 0xFFFF && tbl[H.xbase[s] + cd.hit[s]] == key) ++own;
    const bool keep = own >= 3 || (own >= 2 && cd.nx == 6);
    cd.keep = keep;
    if (keep) kept[atomicAdd(&H.n_kept, 1)] = (uint16_t)c;
  }
  __syncthreads();
  const int nk = H.n_kept;
  unsigned long long* best = tbl;                            // table is dead: reuse for the best u/v keys
  for (int i = tid; i < nk; i += kSeedThreads) best[i] = kNoKey;
  __syncthreads();

  // ---- S4: u/v addition (O8, O9) --------------------------------------------------------------
  {
    const int gl = tid % kUvGroup, gid = tid / kUvGroup, ngroups = kSeedThreads / kUvGroup;
    const unsigned gmask = ((1u << kUvGroup) - 1u) << ((lane / kUvGroup) * kUvGroup);
    for (int w = gid; w < 2 * nk; w += ngroups) {
      const int k = w >> 1, pp = w & 1;
      const Cand& cd = cand[kept[k]];
      float xp[6];
#pragma unroll
      for (int s = 0; s < 6; ++s) xp[s] = xz_at(p, cd.ax, cd.bx, cd.cx, p.ul[s]);
      const int lf = p.uv_first[pp], sf = p.slot_of_layer[lf];
      float xpf = xp[0];
#pragma unroll
      for (int s = 1; s < 6; ++s) xpf = (s == sf) ? xp[s] : xpf;
      const float wa = xpf - p.ywin_a[h][lf], wb = xpf - p.ywin_b[h][lf];
      const float wlo = wa < wb ? wa : wb, whi = wa > wb ? wa : wb;
      const int bf = zl[lf], ef = zl[lf + 1];
      const int first = lower_bound(hx, bf, ef, wlo), last = upper_bound(hx, bf, ef, whi);
      unsigned long long bk = kNoKey;
      for (int ih = first + gl; ih < last; ih += kUvGroup) {
        UvComb c;
        // sf is one of two values per launch; dispatch so that the walk is fully unrolled
        switch (sf) {
          case 0: uv_walk(p, hx, zl, xp, 0, ih, c); break;
          case 1: uv_walk(p, hx, zl, xp, 1, ih, c); break;
          case 2: uv_walk(p, hx, zl, xp, 2, ih, c); break;
          case 3: uv_walk(p, hx, zl, xp, 3, ih, c); break;
          case 4: uv_walk(p, hx, zl, xp, 4, ih, c); break;
          default: uv_walk(p, hx, zl, xp, 5, ih, c); break;
        }
        if (c.n < p.min_uv_hits) continue;
        float ay, by;
        const float chi2y = fit_y(p, c, ay, by);
        if (chi2y > p.chi2y_max) continue;
        const unsigned long long key = ((unsigned long long)(6 - c.n) << 49) |
                                       ((unsigned long long)__float_as_uint(chi2y) << 17) |
                                       ((unsigned long long)pp << 16) | (unsigned long long)(ih - bf);
        bk = key < bk ? key : bk;
      }
#pragma unroll
      for (int o = kUvGroup / 2; o > 0; o >>= 1) {
        const unsigned long long other = __shfl_xor_sync(gmask, bk, o);
        bk = other < bk ? other : bk;
      }
      if (gl == 0 && bk != kNoKey) atomicMin(&best[k], bk);
    }
  }
  __syncthreads();

  // ---- S5: seeds (O10) ------------------------------------------------------------------------
  const int pol = p.pol ? (int)p.pol[event] : p.polarity;
  for (int k = tid; k < nk; k += kSeedThreads) {
    const unsigned long long key = best[k];
    if (key == kNoKey) continue;                             // fake x-z projection (L219)
    const Cand& cd = cand[kept[k]];
    const int pp = (int)(key >> 16) & 1;
    const int lf = p.uv_first[pp], sf = p.slot_of_layer[lf];
    const int ih = zl[lf] + (int)(key & 0xFFFF);
    float xp[6];
#pragma unroll
    for (int s = 0; s < 6; ++s) xp[s] = xz_at(p, cd.ax, cd.bx, cd.cx, p.ul[s]);
    UvComb c;
    switch (sf) {
      case 0: uv_walk(p, hx, zl, xp, 0, ih, c); break;
      case 1: uv_walk(p, hx, zl, xp, 1, ih, c); break;
      case 2: uv_walk(p, hx, zl, xp, 2, ih, c); break;
      case 3: uv_walk(p, hx, zl, xp, 3, ih, c); break;
      case 4: uv_walk(p, hx, zl, xp, 4, ih, c); break;
      default: uv_walk(p, hx, zl, xp, 5, ih, c); break;
    }
    float ay, by;
    const float chi2y = fit_y(p, c, ay, by);
    const int slot = atomicAdd(&H.n_seed, 1);
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
      p.hits[(size_t)lx * ct + o] = cd.hit[s] == 0xFFFF ? LHCB_NO_HIT : a0 + (uint32_t)(zl[lx] + cd.hit[s]);
      p.hits[(size_t)lu * ct + o] = c.hit[s] < 0 ? LHCB_NO_HIT : a0 + (uint32_t)c.hit[s];
    }
    p.nx[o] = cd.nx;
    p.nuv[o] = (uint8_t)c.n;
  }
  __syncthreads();
  if (tid == 0) {
    int ns = H.n_seed;
    unsigned st = H.status;
    if (ns > p.max_seeds) { ns = p.max_seeds; st |= LHCB_ST_SEED_OVERFLOW; }
    p.count[half_id] = (uint32_t)ns;
    p.status[half_id] = st;
  }
}

}  // namespace lhcb
