// VELO-SciFi Matching kernel (section 4) for sm_100a.
//
// One CTA per event.  The event's VELO states are staged in shared memory; the x0 of the event's UT
// hits (four sorted layers, contiguous in memory) is fetched with one bulk async copy that lands while
// the all-pairs loop runs, so the UT searches are shared-memory binary searches.
//   M0     VELO states are counting-sorted into 256 t_y bins in shared memory
//   M1/M2  "all seed x VELO pairs" (L279) without touching most of them: the |dty| cut of Eq. 21 selects
//          a contiguous range of the t_y-binned VELO states (the bins of the window edges, with a safety
//          margin; the literal cut is still applied to every pair in the range, so the accepted set
//          is exactly that of the exhaustive loop).  Thread per seed over its range: kink extrapolation
//          (Eq. 17-18), preselection (Eq. 21); the pairs that pass are queued and a dense pass computes
//          chi2_match (Eq. 22-23) < 2 and writes the pair records
//   M3a    thread per queued pair: loose UT window, layer by layer until one has hits; every such hit
//          becomes a queued hypothesis (Eq. 19-20, Table 2, reading A13)
//   M3b    thread per hypothesis: tight windows in the remaining layers, gamma_x refits; the best
//          hypothesis of each pair wins a packed-key atomicMin (max hits, min residuals, first hit)
//   M4     one-to-one selection with two rounds of 64-bit atomicMin (reading A14); the winning
//          hypothesis of each selected pair is walked once more to write its hits
//
// Arithmetic follows DESIGN.md "Arithmetic specification"; compiled with -fmad=false.
#pragma once
#include <cstdint>

#include "../../include/lhcb.h"
#include "seeding.cuh"   // lower_bound, kNoKey

namespace lhcb {


constexpr int kTyBins = 256;                 // t_y bins of the VELO states (counting sort of M0)

struct MatchParams {
  float zS, zV, dzyS, dzyV, mag[5], presel[4], cx0, cx1, cy0, cy1, inv_tol_tx, inv_tol_ty, chi2m_max;
  float inv_KB, Ag, Bg, inv_Bg, ut_dz[4], ut_dz2[4], ut_dz4[4], ut_tan[4], ut_y_tol;
  float ut_loose[4][4], ut_tight[4][4];
  float row_y0, row_pitch;  // strip row r covers y in [row_y0 + r * row_pitch, that + row_pitch]
  int min_ut_hits, use_ut, polarity;
  int max_seeds, max_long, max_mc, max_velo, max_ut;
  uint32_t n_ut_total;
  // batch
  int n_events;
  const uint32_t* seed_count;
  const float* state;
  size_t seed_cap_total;
  const uint32_t* velo_off;
  const float *vx, *vy, *vtx, *vty;
  const int8_t* pol;
  const uint32_t* ut_off;
  const float *ux, *uylo, *uyhi;
  const uint8_t* urow;      // strip row per UT hit (then uylo / uyhi are not read) or NULL
  uint32_t* count;
  uint32_t* seed_idx;
  uint32_t* velo_idx;
  uint32_t* ut_idx;
  uint8_t* n_ut;
  float* qop;
  float* chi2;
  uint32_t* status;
  size_t long_cap_total;
  // ghost-killing network (reading A14b): packed weights on the device or NULL; seed hit counts; output
  const float* nn;
  const uint8_t *snx, *snuv;
  float* ghost;
  const uint32_t* shits;    // [12][seed_cap_total] hit indices of the seeds or NULL (tie-break of reading A21)
  const uint32_t* order;    // optional CTA -> event map (heaviest events first) or NULL
  const uint32_t* done;     // optional per-half "seeds are in global memory" flags of the Seeding (see SeedParams)
};

struct __align__(8) MatchCand {
  uint16_t seed, velo;      // event-local seed index; rank of the VELO state in t_y order
  float chi2, q0, gamma;    // chi2_match, kick q/p (A10), gamma_x of the best UT hypothesis
  unsigned long long key;   // best UT hypothesis: (4 - n_ut) << 50 | f32 bits of sum res^2 << 18 | layer << 16 | first hit
  uint16_t ut[4];           // its hits, relative to the event's first UT hit (0xFFFF = none)
};
static_assert(sizeof(MatchCand) == 32, "MatchCand is 32 bytes");

// Shared-memory map of one CTA (T threads):
//   [header 64 | UT x0 tile | UT strip rows | VELO states sorted by t_y (x, y, tx, ty) | original index u16 |
//    t_y bin starts u16[257] | scan scratch | region X | pair records | best key per seed | best key per VELO]
// Region X is used in turn as the scatter cursors of M0, the seed states of the current tile (M1/M2), the UT
// hypothesis queue (M3) and the ghost probabilities (M4).  After M3 the UT tile is dead: M4 keeps the network
// weights and the seed states there.
__host__ __device__ inline size_t match_align16(size_t b) { return (b + 15) & ~(size_t)15; }
__host__ __device__ inline size_t match_x_bytes(int T, int max_mc) {
  size_t b = (size_t)T * 16;                                   // float4 per owner of a tile
  if (b < (size_t)kTyBins * 4) b = (size_t)kTyBins * 4;        // scatter cursors
  if (b < (size_t)max_mc * 8) b = (size_t)max_mc * 8;          // 2 * max_mc hypotheses / max_mc ghost probabilities
  return b;
}
__host__ __device__ inline size_t match_ut_bytes(int max_seeds, int max_ut) {
  size_t b = ((size_t)max_ut + 8) * 4;                         // x0 tile (16-byte aligned superset)
  const size_t m4 = 1360 + (size_t)2 * max_seeds * 16;         // M4: network weights + seed states
  return match_align16(b > m4 ? b : m4);
}
__host__ __device__ inline size_t match_smem_bytes(int T, int max_seeds, int max_mc, int max_velo, int max_ut) {
  size_t b = 64;
  b += match_ut_bytes(max_seeds, max_ut);
  b += match_align16((size_t)max_ut + 32);   // strip rows (16-byte aligned superset)
  b += (size_t)max_velo * 16;                // VELO states, sorted by ty
  b += match_align16((size_t)max_velo * 2);  // original index of each sorted state
  b += match_align16((size_t)(kTyBins + 1) * 2);   // start of each t_y bin
  b += 144;                                  // two warp_sums buffers of the block scan
  b += match_align16(match_x_bytes(T, max_mc));
  b += (size_t)max_mc * sizeof(MatchCand);
  b += (size_t)2 * max_seeds * 8;            // best key per seed
  b += (size_t)max_velo * 8;                 // best key per VELO track
  return b;
}

// ---- ghost-killing network (L344-348, reading A14b).  exp and log are spelled out operation by operation
// (DESIGN.md "Arithmetic specification"): no libm, no fast-math intrinsics, -fmad=false.
__device__ __forceinline__ float nn_exp(float y) {
  y = y > 87.f ? 87.f : y;
  y = y < -87.f ? -87.f : y;
  const float n = floorf(y * 1.44269504f + 0.5f);
  const float r = (y - n * 0.693359375f) - n * -2.12194440e-4f;       // Cody-Waite reduction
  float q = 1.0f / 720.0f;
  q = q * r + 1.0f / 120.0f;
  q = q * r + 1.0f / 24.0f;
  q = q * r + 1.0f / 6.0f;
  q = q * r + 0.5f;
  q = q * r + 1.0f;
  q = q * r + 1.0f;
  return q * __int_as_float(((int)n + 127) << 23);                    // times 2^n, |n| <= 126: exact scaling
}
__device__ __forceinline__ float nn_log(float x) {                     // x normal and positive
  const unsigned int b = __float_as_uint(x);
  int e = (int)((b >> 23) & 0xFFu) - 126;
  float m = __uint_as_float((b & 0x807FFFFFu) | 0x3F000000u);          // x = m 2^e, m in [1/2, 1)
  if (m < 0.70710678f) { m = m * 2.0f; e -= 1; }
  const float s = (m - 1.0f) / (m + 1.0f);
  const float s2 = s * s;
  float q = 2.0f / 9.0f;
  q = q * s2 + 2.0f / 7.0f;
  q = q * s2 + 2.0f / 5.0f;
  q = q * s2 + 2.0f / 3.0f;
  q = q * s2 + 2.0f;
  return (float)e * 0.69314718f + s * q;
}
__device__ __forceinline__ float nn_eta(float tx, float ty) {          // pseudorapidity from the slopes
  const float rho2 = tx * tx + ty * ty;
  float rho = sqrtf(rho2);
  const float sh = sqrtf(1.0f + rho2);
  rho = rho < 1e-6f ? 1e-6f : rho;
  return nn_log((1.0f + sh) / rho);
}
// nn = mu[8], isig[8], W1[32][8], b1[32], W2[32], b2, cut, margin (a copy in shared memory: every lane reads
// the same weight, a broadcast)
__device__ __forceinline__ float nn_ghost_prob(const float* __restrict__ nn, const float* in) {
  float u[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) u[k] = (in[k] - nn[k]) * nn[8 + k];
  float t = nn[336];
#pragma unroll 4
  for (int j = 0; j < 32; ++j) {
    float h = nn[272 + j];
#pragma unroll
    for (int k = 0; k < 8; ++k) h = h + nn[16 + j * 8 + k] * u[k];
    h = h < 0.f ? 0.f : h;
    t = t + nn[304 + j] * h;
  }
  return 1.0f / (1.0f + nn_exp(-t));
}

struct UtHyp { int n; int idx[4]; float gamma, ssq; };      // idx: position in the searched x0 array, -1 = none

__device__ __forceinline__ float ut_window(const float* w, float invpG) {
  const float v = w[0] + w[1] * invpG;                      // L315
  const float lo = v > w[2] ? v : w[2];
  return lo < w[3] ? lo : w[3];
}

// Does the strip of UT hit i (index into the searched x0 array) cover y within ut_y_tol (reading A18)?
// Strip rows (one byte per hit, staged in shared memory): y_lo = row_y0 + row * row_pitch, y_hi = y_lo +
// row_pitch, the same float operations that produced the y_lo / y_hi arrays the float form carries.
struct UtCover {
  const uint8_t* __restrict__ row;     // shared-memory rows or NULL
  const float* __restrict__ ylo;       // global arrays (already offset to the indexing of the x0 array)
  const float* __restrict__ yhi;
  float y0, pitch, tol;
  __device__ __forceinline__ bool operator()(int i, float y) const {
    float lo, hi;
    if (row) { lo = y0 + (float)row[i] * pitch; hi = lo + pitch; }
    else { lo = ylo[i]; hi = yhi[i]; }
    return lo - tol <= y && y <= hi + tol;
  }
};

// O13, second half: hypothesis (layer i0, hit j) of one accepted pair.  The remaining layers use tight
// windows and the closest hit; gamma_x is refitted after each hit (L309).  ux is the searched x0 array
// (shared-memory tile or the global array), uo[] its layer offsets.
__device__ __forceinline__ void ut_tight_walk(const MatchParams& p, float xV, float yV, float txV, float tyV,
                                              float invpG, int i0, int j, const float* __restrict__ ux,
                                              const UtCover& cover, const int* uo, UtHyp& hy) {
  float dj[4];
  float num = 0.f, den = 0.f, gam = 0.f;
  hy.n = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    hy.idx[i] = -1; dj[i] = 0.f;
    if (i < i0) continue;
    const float yt = yV + tyV * p.ut_dz[i];
    int bj = -1;
    if (i == i0) {
      bj = j;
    } else {
      const float xt = (xV + txV * p.ut_dz[i]) + gam * p.ut_dz2[i];            // Eq. 19
      const float xe = xt - yt * p.ut_tan[i];
      const float wt = ut_window(p.ut_tight[i], invpG);
      const float tlo = xe - wt, thi = xe + wt;
      const int bb = uo[i], ee = uo[i + 1];
      float bd = 0.f;
      for (int jj = lower_bound(ux, bb, ee, tlo); jj < ee && ux[jj] <= thi; ++jj) {
        if (!cover(jj, yt)) continue;
        const float dd = fabsf(ux[jj] - xe);
        if (bj < 0 || dd < bd) { bj = jj; bd = dd; }
      }
    }
    if (bj >= 0) {
      hy.idx[i] = bj; ++hy.n;
      dj[i] = ((ux[bj] + yt * p.ut_tan[i]) - xV) - txV * p.ut_dz[i];
      if (i == i0) { num = dj[i] * p.ut_dz2[i]; den = p.ut_dz4[i]; }
      else { num = num + dj[i] * p.ut_dz2[i]; den = den + p.ut_dz4[i]; }
      gam = num / den;
    }
  }
  hy.gamma = gam; hy.ssq = 0.f;
  bool first = true;
#pragma unroll
  for (int i = 0; i < 4; ++i)
    if (hy.idx[i] >= 0) {
      const float res = dj[i] - gam * p.ut_dz2[i];
      hy.ssq = first ? res * res : hy.ssq + res * res;
      first = false;
    }
}

// one bulk async copy global -> shared signalling mbar
__device__ __forceinline__ void bulk_copy(void* dst, const void* src, uint32_t bytes, uint32_t mbar_addr) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   (uint32_t)__cvta_generic_to_shared(dst)),
               "l"(src), "r"(bytes), "r"(mbar_addr)
               : "memory");
}

template <int kMatchThreads, int MIN_CTAS>
__global__ void __launch_bounds__(kMatchThreads, MIN_CTAS)
matching_kernel(const __grid_constant__ MatchParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  constexpr int T = kMatchThreads;
  int* hdr = reinterpret_cast<int*>(smem);                  // [0] n_mc, [1] n_long, [2] status, [3] n_hyp, [4..8] UT offsets, [9] tie flag
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + 48);
  size_t off = 64;
  float* sux = reinterpret_cast<float*>(smem + off);                       // UT x0 tile; M4: network weights + seed states
  off += match_ut_bytes(p.max_seeds, p.max_ut);
  uint8_t* srow = smem + off;                                              // UT strip rows
  off += match_align16((size_t)p.max_ut + 32);
  float* svx = reinterpret_cast<float*>(smem + off);
  float* svy = svx + p.max_velo;
  float* svtx = svy + p.max_velo;
  float* svty = svtx + p.max_velo;
  off += (size_t)p.max_velo * 16;
  uint16_t* sorig = reinterpret_cast<uint16_t*>(smem + off);
  off += match_align16((size_t)p.max_velo * 2);
  uint16_t* vbin = reinterpret_cast<uint16_t*>(smem + off);               // [kTyBins + 1]
  off += match_align16((size_t)(kTyBins + 1) * 2);
  int* warp_sums = reinterpret_cast<int*>(smem + off);                    // two buffers of the block scan (M0)
  off += 144;
  unsigned char* regx = smem + off;
  int* vcur = reinterpret_cast<int*>(regx);                                // M0: [kTyBins] scatter cursors
  float4* sown = reinterpret_cast<float4*>(regx);                          // M1/M2: (x, y at z_match_y, tx, ty) of the tile's seeds
  uint32_t* hyq = reinterpret_cast<uint32_t*>(regx);                       // M3: (pair << 18) | (layer << 16) | first hit
  float* sghost = reinterpret_cast<float*>(regx);                          // M4: ghost probability per pair
  const int hyp_cap = (int)(match_x_bytes(T, p.max_mc) / 4);
  off += match_align16(match_x_bytes(T, p.max_mc));
  MatchCand* mc = reinterpret_cast<MatchCand*>(smem + off);
  off += (size_t)p.max_mc * sizeof(MatchCand);
  unsigned long long* seed_best = reinterpret_cast<unsigned long long*>(smem + off);
  unsigned long long* velo_best = seed_best + 2 * p.max_seeds;

  const int tid = threadIdx.x;
  const int e = p.order ? (int)p.order[blockIdx.x] : (int)blockIdx.x;
  int flip = 0;                                            // warp_sums buffer of the next block scan
  LHCB_CLK_INIT
  const uint32_t v0 = p.velo_off[e];
  const int nv = (int)(p.velo_off[e + 1] - v0);
  if (nv > p.max_velo) {
    if (tid == 0) { p.count[e] = 0; p.status[e] = LHCB_ST_VELO_OVERFLOW; }
    return;
  }
  if (tid < 4) hdr[tid] = 0;
  if (tid == 4) { hdr[9] = 0; hdr[10] = 0; hdr[11] = 0; }    // chi2 tie seen (reading A21); preselected pairs of the even / odd tiles
  // ---- UT x0 (and strip rows) of this event: bulk copies, overlapped with the all-pairs loop ----------
  uint32_t u_begin = 0, u_end = 0, ua0 = 0;
  bool ut_in_smem = false, rows_in_smem = false;
  const uint32_t mbar_addr = (uint32_t)__cvta_generic_to_shared(mbar);
  if (p.use_ut) {
    u_begin = p.ut_off[(size_t)e * 4]; u_end = p.ut_off[(size_t)e * 4 + 4];
    if (u_end - u_begin > 65534u) {                          // 16-bit event-local UT indices
      if (tid == 0) { p.count[e] = 0; p.status[e] = LHCB_ST_UT_OVERFLOW; }
      return;
    }
    ua0 = u_begin & ~3u;
    ut_in_smem = (int)(u_end - u_begin) <= p.max_ut;
    rows_in_smem = ut_in_smem && p.urow != nullptr;
    if (ut_in_smem) {
      // x0: floats [ua0, ua1) by one bulk copy, the unaligned tail of the array by plain loads;
      // rows: bytes [ra0, ra1), srow[i - ra0] = row of hit i
      const bool aligned = (reinterpret_cast<uintptr_t>(p.ux) & 15) == 0;
      uint32_t ua1 = (u_end + 3u) & ~3u;
      if (ua1 > (p.n_ut_total & ~3u)) ua1 = p.n_ut_total & ~3u;
      if (!aligned || ua1 < ua0) ua1 = ua0;
      const bool raligned = rows_in_smem && (reinterpret_cast<uintptr_t>(p.urow) & 15) == 0;
      const uint32_t ra0 = u_begin & ~15u;
      uint32_t ra1 = (u_end + 15u) & ~15u;
      if (ra1 > (p.n_ut_total & ~15u)) ra1 = p.n_ut_total & ~15u;
      if (!raligned || ra1 < ra0) ra1 = ra0;
      if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_addr));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const uint32_t bytes = (ua1 - ua0) * 4u + (ra1 - ra0);
        if (bytes > 0) {
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_addr), "r"(bytes) : "memory");
          if (ua1 > ua0) bulk_copy(sux, p.ux + ua0, (ua1 - ua0) * 4u, mbar_addr);
          if (ra1 > ra0) bulk_copy(srow, p.urow + ra0, ra1 - ra0, mbar_addr);
        } else {
          asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar_addr) : "memory");
        }
      }
      for (uint32_t i = (ua1 > u_begin ? ua1 : u_begin) + tid; i < u_end; i += T) sux[i - ua0] = p.ux[i];
      if (rows_in_smem)
        for (uint32_t i = (ra1 > u_begin ? ra1 : u_begin) + tid; i < u_end; i += T) srow[i - ra0] = p.urow[i];
      if (tid < 5) hdr[4 + tid] = (int)(p.ut_off[(size_t)e * 4 + tid] - ua0);
    } else if (tid < 5) {
      hdr[4 + tid] = (int)p.ut_off[(size_t)e * 4 + tid];
    }
  }
  // t_y bin of a VELO state or of a window edge: monotone in t, so the states with t in [a, b] lie in the bins
  // [bin(a), bin(b)] whatever the rounding; values outside +-0.4 land in the edge bins
  auto ty_bin = [](float t) { return (int)fminf(fmaxf((t + 0.4f) * ((float)kTyBins / 0.8f), 0.f), (float)(kTyBins - 1)); };
  for (int v = tid; v < nv; v += T) velo_best[v] = kNoKey;
  for (int b = tid; b < kTyBins; b += T) vcur[b] = 0;
  __syncthreads();
  // ---- M0: counting sort of the VELO states into t_y bins (order inside a bin is irrelevant: the bins
  // only delimit, per seed, a superset of the states that can pass the |dty| cut of Eq. 21) -----------
  for (int v = tid; v < nv; v += T) atomicAdd(&vcur[ty_bin(p.vty[v0 + v])], 1);
  __syncthreads();
  {
    constexpr int per = kTyBins / T;
    static_assert(per * T == kTyBins, "whole bins per thread");
    int c[per], sum = 0;
#pragma unroll
    for (int k = 0; k < per; ++k) { c[k] = vcur[tid * per + k]; sum += c[k]; }
    int total;
    int run = block_exscan<T>(sum, warp_sums, flip, total);
    if (tid == 0) vbin[0] = 0;
#pragma unroll
    for (int k = 0; k < per; ++k) { vcur[tid * per + k] = run; run += c[k]; vbin[tid * per + k + 1] = (uint16_t)run; }
  }
  __syncthreads();
  for (int v = tid; v < nv; v += T) {
    const float t = p.vty[v0 + v];
    const int r = atomicAdd(&vcur[ty_bin(t)], 1);
    LHCB_CHECK_IDX(r, nv);
    svx[r] = p.vx[v0 + v]; svy[r] = p.vy[v0 + v]; svtx[r] = p.vtx[v0 + v]; svty[r] = t;
    sorig[r] = (uint16_t)v;
  }
  __syncthreads();
  LHCB_CLK(9)

  // ---- the seeds of this event: when the Seeding grid may still be running (programmatic dependent launch,
  // lhcb_order's workspace), wait until both of its halves have raised their flag
  if (p.done) {
    if (tid == 0) {
      const uint32_t* f = p.done + 2 * (size_t)e;
      uint32_t a = 0, b = 0;
      for (;;) {
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(a) : "l"(f) : "memory");
        asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(b) : "l"(f + 1) : "memory");
        if (a != 0u && b != 0u) break;
        __nanosleep(256);
      }
    }
    __syncthreads();
  }
  int c0 = (int)p.seed_count[2 * e], c1 = (int)p.seed_count[2 * e + 1];
  if (c0 > p.max_seeds) c0 = p.max_seeds;
  if (c1 > p.max_seeds) c1 = p.max_seeds;
  const int ns = c0 + c1;
  // ---- M1/M2: all seed x VELO pairs (L279), restricted to the |dty| range of each seed ----------
  const size_t sct = p.seed_cap_total;
  uint32_t* pq = reinterpret_cast<uint32_t*>(seed_best);   // preselected pairs of a tile: (owner << 16) | VELO rank
  const int pq_cap = 4 * p.max_seeds;
  auto slot_of = [&](int s) { return s < c0 ? (size_t)(2 * e) * p.max_seeds + s : (size_t)(2 * e + 1) * p.max_seeds + (s - c0); };
  for (int tile0 = 0, par = 0; tile0 < ns; tile0 += T, par ^= 1) {
    // two pair counters taken in turn.  Only a tile's closing barrier lies between its dense pass and the next
    // tile's walk, so a counter cannot be cleared after that barrier without racing the first increments.  Thread 0
    // clears the OTHER counter between the two barriers of each tile instead: its last reader finished before the
    // previous tile's closing barrier, its next writer starts after this tile's
    int* const pq_n = &hdr[10 + par];
    const int nown = ns - tile0 < T ? ns - tile0 : T;
    int cnt = 0, fst = 0;
    if (tid < nown) {
      const size_t slot = slot_of(tile0 + tid);
      const float xS = p.state[slot], yS = p.state[sct + slot], txS = p.state[2 * sct + slot], tyS = p.state[3 * sct + slot];
      sown[tid] = make_float4(xS, yS + p.dzyS * tyS, txS, tyS);                    // L231: y at z_match_y
      // superset of {v : |tyS - tyV| < presel[3]} whatever the rounding of the subtraction
      const float w = p.presel[3] + 1e-6f * (fabsf(tyS) + p.presel[3]) + 1e-30f;
      fst = vbin[ty_bin(tyS - w)];
      const int lst = vbin[ty_bin(tyS + w) + 1];
      cnt = lst - fst;
    }
    LHCB_CLK(10)
    if (tid < nown) {                                        // thread per seed: its own range of VELO states
      const float4 o = sown[tid];
      const float xS = o.x, ys = o.y, txS = o.z, tyS = o.w, axS = fabsf(xS);
      LHCB_CHECK_IDX(fst + cnt, nv + 1);
      for (int v = fst; v < fst + cnt; ++v) {
        const float xV = svx[v], yV = svy[v], txV = svtx[v], tyV = svty[v];
        const float dtx = txS - txV, dty = tyS - tyV, adtx = fabsf(dtx);
        const float zm = (((p.mag[0] + p.mag[1] * adtx) + p.mag[2] * (dtx * dtx)) + p.mag[3] * axS) +
                         p.mag[4] * (txV * txV);                                   // Eq. 18
        const float xs = xS + (zm - p.zS) * txS, xv = xV + (zm - p.zV) * txV;      // Eq. 17
        const float yv = yV + p.dzyV * tyV;
        const float dx = xs - xv, dy = ys - yv;
        if (!(fabsf(dx) < p.presel[0] && fabsf(dy) < p.presel[1] && adtx < p.presel[2] &&
              fabsf(dty) < p.presel[3]))                                           // Eq. 21
          continue;
        const int k = smem_inc(pq_n);
        if (k < pq_cap) pq[k] = ((uint32_t)tid << 16) | (uint32_t)v;
      }
    }
    __syncthreads();
    int nq = *pq_n;
    if (tid == 0) hdr[10 + (par ^ 1)] = 0;                   // the next tile's counter: idle since before the previous closing barrier
    if (nq > pq_cap) { nq = pq_cap; if (tid == 0) hdr[2] |= LHCB_ST_MATCH_OVERFLOW; }
    for (int i = tid; i < nq; i += T) {
      const uint32_t e_ = pq[i];
      const int t = (int)(e_ >> 16), v = (int)(e_ & 0xFFFFu);
      const float4 o = sown[t];
      const float xS = o.x, ys = o.y, txS = o.z, tyS = o.w;
      const float xV = svx[v], yV = svy[v], txV = svtx[v], tyV = svty[v];
      // the same operations on the same operands as in the walk above: the same values
      const float dtx = txS - txV, dty = tyS - tyV, adtx = fabsf(dtx);
      const float zm = (((p.mag[0] + p.mag[1] * adtx) + p.mag[2] * (dtx * dtx)) + p.mag[3] * fabsf(xS)) +
                       p.mag[4] * (txV * txV);                                   // Eq. 18
      const float xs = xS + (zm - p.zS) * txS, xv = xV + (zm - p.zV) * txV;      // Eq. 17
      const float yv = yV + p.dzyV * tyV;
      const float dx = xs - xv, dy = ys - yv;
      const float tolx = p.cx0 + p.cx1 * (dtx * dtx);                            // Eq. 23
      const float toly = p.cy0 + p.cy1 * (txV * txV + tyV * tyV);
      const float chi2 = (((dx * dx) / tolx + (dy * dy) / toly) + (dtx * dtx) * p.inv_tol_tx) +
                         (dty * dty) * p.inv_tol_ty;                             // Eq. 22
      if (!(chi2 < p.chi2m_max)) continue;                                       // L301
      const int k = smem_inc(&hdr[0]);
      if (k < p.max_mc) {
        MatchCand m;
        m.seed = (uint16_t)(tile0 + t); m.velo = (uint16_t)v; m.chi2 = chi2; m.q0 = dtx * p.inv_KB;   // A10
        m.gamma = 0.f; m.key = kNoKey;
#pragma unroll
        for (int l = 0; l < 4; ++l) m.ut[l] = 0xFFFF;
        mc[k] = m;
      }
    }
    __syncthreads();
    LHCB_CLK(11)
  }
  for (int s = tid; s < 2 * p.max_seeds; s += T) seed_best[s] = kNoKey;   // (the queue of preselected pairs is dead)
  __syncthreads();                                         // without UT and without a network nothing else separates this reset
                                                           // from the atomicMin of the selection below
  int nm = hdr[0];
  LHCB_DBG_MAX(4, nm)
  if (nm > p.max_mc) { nm = p.max_mc; if (tid == 0) hdr[2] |= LHCB_ST_MATCH_OVERFLOW; }

  // ---- M3: UT hits (O13) -----------------------------------------------------------------------
  if (ut_in_smem) {
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
  LHCB_CLK(14)
  // searched x0 array (shared tile or global), its y coverage, and the index of its element 0 relative to
  // the event's first UT hit
  const float* __restrict__ ux = ut_in_smem ? sux : p.ux;
  const int rel0 = ut_in_smem ? (int)(ua0 - u_begin) : -(int)u_begin;
  UtCover cover;
  cover.row = rows_in_smem ? srow + (ua0 - (u_begin & ~15u)) : nullptr;             // row of x0-tile element i at cover.row[i]
  cover.ylo = p.urow ? nullptr : p.uylo + (ut_in_smem ? ua0 : 0u);
  cover.yhi = p.urow ? nullptr : p.uyhi + (ut_in_smem ? ua0 : 0u);
  cover.y0 = p.row_y0; cover.pitch = p.row_pitch; cover.tol = p.ut_y_tol;
  if (p.urow && !rows_in_smem) cover.row = p.urow + (ut_in_smem ? ua0 : 0u);       // event too large for the tile: rows from global memory
  const int* uo = hdr + 4;
  if (p.use_ut) {
    // M3a: loose windows, layer by layer until one has hits; each hit is a hypothesis (A13)
    for (int k = tid; k < nm; k += T) {
      MatchCand& m = mc[k];
      const int v = m.velo;
      const float xV = svx[v], yV = svy[v], txV = svtx[v], tyV = svty[v], q0 = m.q0;
      const float invpG = fabsf(q0) * 1000.f;
      const float gamma0 = p.Ag + p.Bg * q0;                                      // Eq. 20
      bool found = false;
      for (int i0 = 0; i0 < 4 && !found; ++i0) {
        if (4 - i0 < p.min_ut_hits) break;
        const float yi = yV + tyV * p.ut_dz[i0];
        const float xi = (xV + txV * p.ut_dz[i0]) + gamma0 * p.ut_dz2[i0];        // Eq. 19
        const float x0e = xi - yi * p.ut_tan[i0];
        const float w = ut_window(p.ut_loose[i0], invpG);
        const float lo = x0e - w, hi = x0e + w;
        const int b = uo[i0], ee = uo[i0 + 1];
        for (int j = lower_bound(ux, b, ee, lo); j < ee && ux[j] <= hi; ++j) {
          if (ut_in_smem) LHCB_CHECK_IDX(j, p.max_ut + 8);
          if (!cover(j, yi)) continue;
          found = true;
          const int slot = smem_inc(&hdr[3]);
          if (slot < hyp_cap) hyq[slot] = ((uint32_t)k << 18) | ((uint32_t)i0 << 16) | (uint32_t)(j + rel0);
        }
      }
    }
    __syncthreads();
    int nh = hdr[3];
    LHCB_DBG_MAX(5, nh)
    if (nh > hyp_cap) { nh = hyp_cap; if (tid == 0) hdr[2] |= LHCB_ST_MATCH_OVERFLOW; }
    // M3b: tight walk of every hypothesis; the best one of each pair wins the atomicMin and, after the
    // barrier, leaves its hits and gamma_x in the pair's record (a better hypothesis of a later round
    // overwrites them)
    for (int i0r = 0; i0r < nh; i0r += T) {
      const int i = i0r + tid;
      UtHyp hy;
      unsigned long long key = kNoKey;
      int k = 0;
      if (i < nh) {
        const uint32_t hq = hyq[i];
        k = (int)(hq >> 18);
        const int i0 = (int)((hq >> 16) & 3u), jrel = (int)(hq & 0xFFFFu);
        const MatchCand& m = mc[k];
        const int v = m.velo;
        ut_tight_walk(p, svx[v], svy[v], svtx[v], svty[v], fabsf(m.q0) * 1000.f, i0, jrel - rel0, ux, cover, uo, hy);
        key = ((unsigned long long)(4 - hy.n) << 50) | ((unsigned long long)__float_as_uint(hy.ssq) << 18) |
              (hq & 0x3FFFFu);
        LHCB_CHECK_IDX(k, nm);
        atomicMin(&mc[k].key, key);
      }
      __syncthreads();
      if (i < nh && mc[k].key == key) {
        MatchCand& m = mc[k];
        m.gamma = hy.gamma;
#pragma unroll
        for (int l = 0; l < 4; ++l) m.ut[l] = hy.idx[l] < 0 ? (uint16_t)0xFFFF : (uint16_t)(hy.idx[l] + rel0);
      }
    }
    __syncthreads();
  }
  LHCB_CLK(12)
  // a pair is valid if its best hypothesis has enough UT hits (L311); without UT every pair is
  const unsigned long long key_ok = p.use_ut ? (unsigned long long)(4 - p.min_ut_hits) : ~0ull >> 50;
  const bool use_nn = p.nn != nullptr;
  float nn_cut = 0.f, nn_margin = 0.f;
  if (use_nn) {
    // ---- M4 (O14b, L346-348): ghost probability of every valid pair; minimum per seed and per VELO over
    // the pairs below the cut.  The UT tile is dead: the network and the seed states are staged over it.
    float* snn = sux;                                                              // [339] (+ padding to 340)
    float4* sst = reinterpret_cast<float4*>(sux + 340);                            // [ns] x, y, tx, ty
    for (int i = tid; i < LHCB_GHOST_NN_SIZE; i += T) snn[i] = __ldg(p.nn + i);
    for (int s = tid; s < ns; s += T) {
      const size_t slot = slot_of(s);
      sst[s] = make_float4(p.state[slot], p.state[sct + slot], p.state[2 * sct + slot], p.state[3 * sct + slot]);
    }
    __syncthreads();
    nn_cut = snn[337]; nn_margin = snn[338];
    for (int k = tid; k < nm; k += T) {
      const MatchCand& m = mc[k];
      if ((m.key >> 50) > key_ok) continue;
      const int s = m.seed, v = m.velo;
      const float4 st = sst[s];
      const float xS = st.x, yS = st.y, txS = st.z, tyS = st.w;
      const float xV = svx[v], yV = svy[v], txV = svtx[v], tyV = svty[v];
      const float dtx = txS - txV, dty = tyS - tyV, adtx = fabsf(dtx);
      const float zm = (((p.mag[0] + p.mag[1] * adtx) + p.mag[2] * (dtx * dtx)) + p.mag[3] * fabsf(xS)) +
                       p.mag[4] * (txV * txV);                                     // Eq. 18
      const float xs = xS + (zm - p.zS) * txS, xv = xV + (zm - p.zV) * txV;        // Eq. 17
      const float ys = yS + p.dzyS * tyS, yv = yV + p.dzyV * tyV;
      float in[8];
      in[0] = zm; in[1] = xs - xv; in[2] = ys - yv; in[3] = dtx; in[4] = dty; in[5] = m.chi2;
      in[6] = nn_eta(txV, tyV);
      const size_t slot = slot_of(s);
      in[7] = (float)(p.snx && p.snuv ? (int)p.snx[slot] + (int)p.snuv[slot] : 12);
      const float g = nn_ghost_prob(snn, in);
      sghost[k] = g;
      if (g < nn_cut) {
        atomicMin(&seed_best[s], (unsigned long long)__float_as_uint(g));
        atomicMin(&velo_best[sorig[v]], (unsigned long long)__float_as_uint(g));
      }
    }
    __syncthreads();
  } else {
  for (int k = tid; k < nm; k += T) {
    const MatchCand& m = mc[k];
    LHCB_CHECK_IDX(m.seed, ns); LHCB_CHECK_IDX(sorig[m.velo], nv);
    if ((m.key >> 50) <= key_ok)
      atomicMin(&seed_best[m.seed], ((unsigned long long)__float_as_uint(m.chi2) << 32) | sorig[m.velo]);
  }
  __syncthreads();
  // ---- M4: one-to-one selection (O14) -------------------------------------------------------------
  for (int k = tid; k < nm; k += T) {
    const MatchCand& m = mc[k];
    if ((m.key >> 50) > key_ok) continue;
    const unsigned long long cb = (unsigned long long)__float_as_uint(m.chi2) << 32;
    if (seed_best[m.seed] != (cb | sorig[m.velo])) continue;
    const unsigned long long old = atomicMin(&velo_best[sorig[m.velo]], cb | m.seed);
    // Reading A21: an exact chi2 tie between two seeds for one VELO state (twin seeds: bit-identical states
    // from duplicate hits) is decided by the seeds' hit lists, not by their slot order.  Whoever meets a
    // different seed at its own chi2 reports the tie; the (rare) event that has one resolves it serially.
    if ((old >> 32) == (cb >> 32) && (uint32_t)old != (uint32_t)m.seed) hdr[9] = 1;
  }
  __syncthreads();
  if (hdr[9]) {
    if (tid == 0) {
      auto before = [&](int a, int b) {                        // hit lists in lexicographic order, then the index
        if (p.shits)
          for (int l = 0; l < 12; ++l) {
            const uint32_t ha = p.shits[(size_t)l * sct + slot_of(a)], hb = p.shits[(size_t)l * sct + slot_of(b)];
            if (ha != hb) return ha < hb;
          }
        return a < b;
      };
      for (int k = 0; k < nm; ++k) {
        const MatchCand& m = mc[k];
        if ((m.key >> 50) > key_ok) continue;
        const unsigned long long cb = (unsigned long long)__float_as_uint(m.chi2) << 32;
        if (seed_best[m.seed] != (cb | sorig[m.velo])) continue;
        const unsigned long long vb = velo_best[sorig[m.velo]];
        if ((vb >> 32) == (cb >> 32) && before((int)m.seed, (int)(uint32_t)vb)) velo_best[sorig[m.velo]] = cb | m.seed;
      }
    }
    __syncthreads();
  }
  }
  const int pol = p.pol ? (int)p.pol[e] : p.polarity;
  for (int k = tid; k < nm; k += T) {
    const MatchCand& m = mc[k];
    if ((m.key >> 50) > key_ok) continue;
    const unsigned long long cb = (unsigned long long)__float_as_uint(m.chi2) << 32;
    const int vo = sorig[m.velo];
    float g = 0.f;
    if (use_nn) {
      // kept if below the cut and no track sharing its seed or its VELO is better by the margin (the minimum
      // includes the track itself, which never satisfies g >= g + margin)
      g = sghost[k];
      if (!(g < nn_cut)) continue;
      const float gs = __uint_as_float((unsigned int)seed_best[m.seed]), gv = __uint_as_float((unsigned int)velo_best[vo]);
      if (g >= gs + nn_margin || g >= gv + nn_margin) continue;
    } else if (seed_best[m.seed] != (cb | vo) || velo_best[vo] != (cb | m.seed)) continue;
    const int slot = smem_inc(&hdr[1]);
    if (slot >= p.max_long) continue;
    const size_t o = (size_t)e * p.max_long + slot, ct = p.long_cap_total;
    p.seed_idx[o] = (uint32_t)slot_of(m.seed);
    p.velo_idx[o] = v0 + vo;
    float q = m.q0;                                                              // A10
    if (p.use_ut) {
#pragma unroll
      for (int l = 0; l < 4; ++l)
        p.ut_idx[(size_t)l * ct + o] = m.ut[l] == 0xFFFF ? LHCB_NO_HIT : u_begin + (uint32_t)m.ut[l];
      p.n_ut[o] = (uint8_t)(4 - (int)(m.key >> 50));
      q = (m.gamma - p.Ag) * p.inv_Bg;                                           // Eq. 20 inverted
    } else {
#pragma unroll
      for (int l = 0; l < 4; ++l) p.ut_idx[(size_t)l * ct + o] = LHCB_NO_HIT;
      p.n_ut[o] = 0;
    }
    p.qop[o] = pol > 0 ? q : -q;
    p.chi2[o] = m.chi2;
    if (use_nn && p.ghost) p.ghost[o] = g;
  }
  __syncthreads();
  LHCB_CLK(13)
  if (tid == 0) {
    int nl = hdr[1];
    unsigned st = (unsigned)hdr[2];
    if (nl > p.max_long) { nl = p.max_long; st |= LHCB_ST_LONG_OVERFLOW; }
    p.count[e] = (uint32_t)nl;
    p.status[e] = st;
  }
}

}  // namespace lhcb
