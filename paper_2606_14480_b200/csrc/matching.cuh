// VELO-SciFi Matching kernel (section 4) for sm_100a.
//
// One CTA per event.  The event's VELO states are staged in shared memory; the x0 of the event's UT
// hits (four sorted layers, contiguous in memory) is fetched with one bulk async copy that lands while
// the all-pairs loop runs, so the UT searches are shared-memory binary searches.
//   M0     VELO states are counting-sorted into 256 t_y bins in shared memory
//   M1/M2  "all seed x VELO pairs" (L279) without touching most of them: the |dty| cut of Eq. 21 selects
//          a contiguous range of the t_y-binned VELO states (the bins of the window edges, with a safety
//          margin; the literal cut is still applied to every pair in the range, so the accepted set
//          is exactly that of the exhaustive loop).  Pairs in range are flattened over the CTA:
//          kink extrapolation (Eq. 17-18), preselection (Eq. 21), chi2_match (Eq. 22-23) < 2; accepted
//          pairs are queued in shared memory
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
};

struct __align__(8) MatchCand {
  uint16_t seed, velo;      // event-local seed index; rank of the VELO state in t_y order
  float chi2, q0, gamma;    // chi2_match, kick q/p (A10), gamma_x of the best UT hypothesis
  unsigned long long key;   // best UT hypothesis: (4 - n_ut) << 50 | f32 bits of sum res^2 << 18 | layer << 16 | first hit
  uint16_t ut[4];           // its hits, relative to the event's first UT hit (0xFFFF = none)
  float ghost;              // ghost probability (network set) 
  uint32_t pad;
};
static_assert(sizeof(MatchCand) == 40, "MatchCand is 40 bytes");

__host__ __device__ inline size_t match_smem_bytes(int kMatchThreads, int max_seeds, int max_mc, int max_velo, int max_ut) {
  size_t b = 64;
  b += ((size_t)max_ut + 8) * 4;             // UT x0 tile (16-byte aligned superset)
  b += (size_t)max_velo * 16;                // VELO states, sorted by ty
  b += (size_t)(kTyBins + 1) * 4;            // start of each t_y bin of the VELO states
  b += (size_t)max_velo * 2;                 // original index of each sorted state
  b = (b + 15) & ~(size_t)15;
  b += (kMatchThreads + 1) * 4 + kMatchThreads * 2 + 64;   // work-list scan scratch
  b = (b + 15) & ~(size_t)15;
  b += (size_t)max_mc * sizeof(MatchCand);
  b += (size_t)max_mc * 4;                   // UT hypothesis queue
  b = (b + 15) & ~(size_t)15;
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
// nn = mu[8], isig[8], W1[32][8], b1[32], W2[32], b2, cut, margin
__device__ __forceinline__ float nn_ghost_prob(const float* __restrict__ nn, const float* in) {
  float u[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) u[k] = (in[k] - __ldg(nn + k)) * __ldg(nn + 8 + k);
  float t = __ldg(nn + 336);
  for (int j = 0; j < 32; ++j) {
    float h = __ldg(nn + 272 + j);
#pragma unroll
    for (int k = 0; k < 8; ++k) h = h + __ldg(nn + 16 + j * 8 + k) * u[k];
    h = h < 0.f ? 0.f : h;
    t = t + __ldg(nn + 304 + j) * h;
  }
  return 1.0f / (1.0f + nn_exp(-t));
}

struct UtHyp { int n; int idx[4]; float gamma, ssq; };      // idx: position in the searched x0 array, -1 = none

__device__ __forceinline__ float ut_window(const float* w, float invpG) {
  const float v = w[0] + w[1] * invpG;                      // L315
  const float lo = v > w[2] ? v : w[2];
  return lo < w[3] ? lo : w[3];
}

// O13, second half: hypothesis (layer i0, hit j) of one accepted pair.  The remaining layers use tight
// windows and the closest hit; gamma_x is refitted after each hit (L309).  ux is the searched x0 array
// (shared-memory tile or the global array), uo[] its layer offsets; the y-range of hit i of ux is
// (uylo[i], uyhi[i]) (global memory, already offset to the indexing of ux).
__device__ __forceinline__ void ut_tight_walk(const MatchParams& p, float xV, float yV, float txV, float tyV,
                                              float invpG, int i0, int j, const float* __restrict__ ux,
                                              const float* __restrict__ uylo, const float* __restrict__ uyhi,
                                              const int* uo, UtHyp& hy) {
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
        if (!(uylo[jj] - p.ut_y_tol <= yt && yt <= uyhi[jj] + p.ut_y_tol)) continue;
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

template <int kMatchThreads, int MIN_CTAS>
__global__ void __launch_bounds__(kMatchThreads, MIN_CTAS)
matching_kernel(const __grid_constant__ MatchParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  int* hdr = reinterpret_cast<int*>(smem);                  // [0] n_mc, [1] n_long, [2] status, [3] n_hyp, [4..8] UT offsets, [9] tie flag
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(smem + 48);
  float* sux = reinterpret_cast<float*>(smem + 64);
  float* svx = sux + p.max_ut + 8;
  float* svy = svx + p.max_velo;
  float* svtx = svy + p.max_velo;
  float* svty = svtx + p.max_velo;
  int* vbin = reinterpret_cast<int*>(svty + p.max_velo);                  // [kTyBins + 1]
  uint16_t* sorig = reinterpret_cast<uint16_t*>(vbin + kTyBins + 1);
  size_t off = 64 + ((size_t)p.max_ut + 8) * 4 + (size_t)p.max_velo * 18 + (size_t)(kTyBins + 1) * 4;
  off = (off + 15) & ~(size_t)15;
  int* offs = reinterpret_cast<int*>(smem + off);                         // [kMatchThreads + 1]
  uint16_t* firsts = reinterpret_cast<uint16_t*>(offs + kMatchThreads + 1);
  int* warp_sums = reinterpret_cast<int*>(smem + off + (kMatchThreads + 1) * 4 + kMatchThreads * 2);
  off += (kMatchThreads + 1) * 4 + kMatchThreads * 2 + 64;
  off = (off + 15) & ~(size_t)15;
  MatchCand* mc = reinterpret_cast<MatchCand*>(smem + off);
  off += (size_t)p.max_mc * sizeof(MatchCand);
  uint32_t* hyq = reinterpret_cast<uint32_t*>(smem + off);                 // (pair << 18) | (layer << 16) | first hit
  off += (size_t)p.max_mc * 4;
  off = (off + 15) & ~(size_t)15;
  unsigned long long* seed_best = reinterpret_cast<unsigned long long*>(smem + off);
  unsigned long long* velo_best = seed_best + 2 * p.max_seeds;

  const int tid = threadIdx.x;
  const int e = blockIdx.x;
  LHCB_CLK_INIT
  const uint32_t v0 = p.velo_off[e];
  const int nv = (int)(p.velo_off[e + 1] - v0);
  int c0 = (int)p.seed_count[2 * e], c1 = (int)p.seed_count[2 * e + 1];
  if (c0 > p.max_seeds) c0 = p.max_seeds;
  if (c1 > p.max_seeds) c1 = p.max_seeds;
  const int ns = c0 + c1;
  if (nv > p.max_velo) {
    if (tid == 0) { p.count[e] = 0; p.status[e] = LHCB_ST_VELO_OVERFLOW; }
    return;
  }
  if (tid < 4) hdr[tid] = 0;
  if (tid == 4) hdr[9] = 0;                                  // chi2 tie seen (reading A21)
  // ---- UT x0 of this event: one bulk copy, overlapped with the all-pairs loop -----------------
  uint32_t u_begin = 0, u_end = 0, ua0 = 0, ua1 = 0;
  bool ut_in_smem = false;
  const uint32_t mbar_addr = (uint32_t)__cvta_generic_to_shared(mbar);
  if (p.use_ut) {
    u_begin = p.ut_off[(size_t)e * 4]; u_end = p.ut_off[(size_t)e * 4 + 4];
    if (u_end - u_begin > 65534u) {                          // 16-bit event-local UT indices
      if (tid == 0) { p.count[e] = 0; p.status[e] = LHCB_ST_UT_OVERFLOW; }
      return;
    }
    ua0 = u_begin & ~3u;
    ut_in_smem = (int)(u_end - u_begin) <= p.max_ut;
    if (ut_in_smem) {
      const bool aligned = (reinterpret_cast<uintptr_t>(p.ux) & 15) == 0;
      ua1 = (u_end + 3u) & ~3u;
      if (ua1 > (p.n_ut_total & ~3u)) ua1 = p.n_ut_total & ~3u;
      if (!aligned || ua1 < ua0) ua1 = ua0;
      if (tid == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbar_addr));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        const uint32_t bytes = (ua1 - ua0) * 4u;
        if (bytes > 0) {
          asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(mbar_addr), "r"(bytes) : "memory");
          asm volatile(
              "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                  (uint32_t)__cvta_generic_to_shared(sux)),
              "l"(p.ux + ua0), "r"(bytes), "r"(mbar_addr)
              : "memory");
        } else {
          asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(mbar_addr) : "memory");
        }
      }
      if (tid == 32 && aligned && ua1 > ua0 && ((reinterpret_cast<uintptr_t>(p.uylo) | reinterpret_cast<uintptr_t>(p.uyhi)) & 15) == 0) {
        // the y ranges of the hits the UT search will touch: pull the event's slice into L2 while M0-M2 run
        const uint32_t bytes = (ua1 - ua0) * 4u;
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p.uylo + ua0), "r"(bytes) : "memory");
        asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p.uyhi + ua0), "r"(bytes) : "memory");
      }
      for (uint32_t i = ua1 + tid; i < u_end; i += kMatchThreads) sux[i - ua0] = p.ux[i];
      if (tid < 5) hdr[4 + tid] = (int)(p.ut_off[(size_t)e * 4 + tid] - ua0);
    } else if (tid < 5) {
      hdr[4 + tid] = (int)p.ut_off[(size_t)e * 4 + tid];
    }
  }
  // t_y bin of a VELO state or of a window edge: monotone in t, so the states with t in [a, b] lie in the bins
  // [bin(a), bin(b)] whatever the rounding; values outside +-0.4 land in the edge bins
  auto ty_bin = [](float t) { return (int)fminf(fmaxf((t + 0.4f) * ((float)kTyBins / 0.8f), 0.f), (float)(kTyBins - 1)); };
  int* vcur = reinterpret_cast<int*>(hyq);                                 // [kTyBins] scatter cursors (hyq is free until M3)
  for (int v = tid; v < nv; v += kMatchThreads) velo_best[v] = kNoKey;
  for (int s = tid; s < ns; s += kMatchThreads) seed_best[s] = kNoKey;
  for (int b = tid; b <= kTyBins; b += kMatchThreads) vbin[b] = 0;
  __syncthreads();
  // ---- M0: counting sort of the VELO states into t_y bins (order inside a bin is irrelevant: the bins
  // only delimit, per seed, a superset of the states that can pass the |dty| cut of Eq. 21) -----------
  for (int v = tid; v < nv; v += kMatchThreads) atomicAdd(&vbin[ty_bin(p.vty[v0 + v]) + 1], 1);
  __syncthreads();
  {
    constexpr int per = kTyBins / kMatchThreads;
    static_assert(per * kMatchThreads == kTyBins, "whole bins per thread");
    int c[per], sum = 0;
#pragma unroll
    for (int k = 0; k < per; ++k) { c[k] = vbin[tid * per + k + 1]; sum += c[k]; }
    int total;
    int run = block_exscan<kMatchThreads>(sum, warp_sums, total);
#pragma unroll
    for (int k = 0; k < per; ++k) { vcur[tid * per + k] = run; run += c[k]; vbin[tid * per + k + 1] = run; }
  }
  __syncthreads();
  for (int v = tid; v < nv; v += kMatchThreads) {
    const float t = p.vty[v0 + v];
    const int r = atomicAdd(&vcur[ty_bin(t)], 1);
    svx[r] = p.vx[v0 + v]; svy[r] = p.vy[v0 + v]; svtx[r] = p.vtx[v0 + v]; svty[r] = t;
    sorig[r] = (uint16_t)v;
  }
  __syncthreads();
  LHCB_CLK(9)

  // ---- M1/M2: all seed x VELO pairs (L279), restricted to the |dty| range of each seed ----------
  const size_t sct = p.seed_cap_total;
  constexpr int T = kMatchThreads;
  for (int tile0 = 0; tile0 < ns; tile0 += T) {
    const int nown = ns - tile0 < T ? ns - tile0 : T;
    int cnt = 0, fst = 0;
    if (tid < nown) {
      const int s = tile0 + tid;
      const size_t slot = s < c0 ? (size_t)(2 * e) * p.max_seeds + s : (size_t)(2 * e + 1) * p.max_seeds + (s - c0);
      const float tyS = p.state[3 * sct + slot];
      // superset of {v : |tyS - tyV| < presel[3]} whatever the rounding of the subtraction
      const float w = p.presel[3] + 1e-6f * (fabsf(tyS) + p.presel[3]) + 1e-30f;
      fst = vbin[ty_bin(tyS - w)];
      const int lst = vbin[ty_bin(tyS + w) + 1];
      cnt = lst - fst;
    }
    int total;
    const int ex = block_exscan<T>(cnt, warp_sums, total);
    offs[tid] = ex; firsts[tid] = (uint16_t)fst;
    if (tid == T - 1) offs[T] = total;
    __syncthreads();
    LHCB_CLK(10)
    const int chunk = (total + T - 1) / T;
    const int p0 = tid * chunk, p1 = p0 + chunk < total ? p0 + chunk : total;
    if (p0 < p1) {
      int t = owner_of(offs, nown, p0) - 1;
      int nxt = -1, f = 0, s = 0;
      float xS = 0.f, txS = 0.f, tyS = 0.f, axS = 0.f, ys = 0.f;
      for (int q = p0; q < p1; ++q) {
        if (q >= nxt) {
          do { ++t; nxt = offs[t + 1]; } while (q >= nxt);
          s = tile0 + t;
          const size_t slot = s < c0 ? (size_t)(2 * e) * p.max_seeds + s : (size_t)(2 * e + 1) * p.max_seeds + (s - c0);
          xS = p.state[slot]; const float yS = p.state[sct + slot]; txS = p.state[2 * sct + slot];
          tyS = p.state[3 * sct + slot];
          axS = fabsf(xS);
          ys = yS + p.dzyS * tyS;                                                  // L231
          f = (int)firsts[t] - offs[t];
        }
        const int v = f + q;                                                       // rank in ty order
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
        const float tolx = p.cx0 + p.cx1 * (dtx * dtx);                            // Eq. 23
        const float toly = p.cy0 + p.cy1 * (txV * txV + tyV * tyV);
        const float chi2 = (((dx * dx) / tolx + (dy * dy) / toly) + (dtx * dtx) * p.inv_tol_tx) +
                           (dty * dty) * p.inv_tol_ty;                             // Eq. 22
        if (!(chi2 < p.chi2m_max)) continue;                                       // L301
        const int k = atomicAdd(&hdr[0], 1);
        if (k < p.max_mc) {
          MatchCand m;
          m.seed = (uint16_t)s; m.velo = (uint16_t)v; m.chi2 = chi2; m.q0 = dtx * p.inv_KB;   // A10
          m.gamma = 0.f; m.key = kNoKey; m.ghost = 0.f; m.pad = 0u;
#pragma unroll
          for (int l = 0; l < 4; ++l) m.ut[l] = 0xFFFF;
          mc[k] = m;
        }
      }
    }
    __syncthreads();
    LHCB_CLK(11)
  }
  __syncthreads();
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
  // searched x0 array (shared tile or global), its y ranges, and the index of its element 0 relative to
  // the event's first UT hit
  const float* __restrict__ ux = ut_in_smem ? sux : p.ux;
  const float* __restrict__ uylo = p.uylo + (ut_in_smem ? ua0 : 0u);
  const float* __restrict__ uyhi = p.uyhi + (ut_in_smem ? ua0 : 0u);
  const int rel0 = ut_in_smem ? (int)(ua0 - u_begin) : -(int)u_begin;
  const int* uo = hdr + 4;
  if (p.use_ut) {
    // M3a: loose windows, layer by layer until one has hits; each hit is a hypothesis (A13)
    for (int k = tid; k < nm; k += kMatchThreads) {
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
          if (!(uylo[j] - p.ut_y_tol <= yi && yi <= uyhi[j] + p.ut_y_tol)) continue;
          found = true;
          const int slot = atomicAdd(&hdr[3], 1);
          if (slot < p.max_mc) hyq[slot] = ((uint32_t)k << 18) | ((uint32_t)i0 << 16) | (uint32_t)(j + rel0);
        }
      }
    }
    __syncthreads();
    int nh = hdr[3];
    LHCB_DBG_MAX(5, nh)
    if (nh > p.max_mc) { nh = p.max_mc; if (tid == 0) hdr[2] |= LHCB_ST_MATCH_OVERFLOW; }
    // M3b: tight walk of every hypothesis; the best one of each pair wins the atomicMin and, after the
    // barrier, leaves its hits and gamma_x in the pair's record (a better hypothesis of a later round
    // overwrites them)
    for (int i0r = 0; i0r < nh; i0r += kMatchThreads) {
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
        ut_tight_walk(p, svx[v], svy[v], svtx[v], svty[v], fabsf(m.q0) * 1000.f, i0, jrel - rel0, ux, uylo, uyhi, uo, hy);
        key = ((unsigned long long)(4 - hy.n) << 50) | ((unsigned long long)__float_as_uint(hy.ssq) << 18) |
              (hq & 0x3FFFFu);
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
  // a pair is valid if its best hypothesis has enough UT hits (L311); without UT every pair is
  const unsigned long long key_ok = p.use_ut ? (unsigned long long)(4 - p.min_ut_hits) : ~0ull >> 50;
  const bool use_nn = p.nn != nullptr;
  float nn_cut = 0.f, nn_margin = 0.f;
  if (use_nn) {
    // ---- M4 (O14b, L346-348): ghost probability of every valid pair; minimum per seed and per VELO over
    // the pairs below the cut
    nn_cut = __ldg(p.nn + 337); nn_margin = __ldg(p.nn + 338);
    for (int k = tid; k < nm; k += kMatchThreads) {
      MatchCand& m = mc[k];
      if ((m.key >> 50) > key_ok) continue;
      const int s = m.seed, v = m.velo;
      const size_t slot = s < c0 ? (size_t)(2 * e) * p.max_seeds + s : (size_t)(2 * e + 1) * p.max_seeds + (s - c0);
      const float xS = p.state[slot], yS = p.state[sct + slot], txS = p.state[2 * sct + slot], tyS = p.state[3 * sct + slot];
      const float xV = svx[v], yV = svy[v], txV = svtx[v], tyV = svty[v];
      const float dtx = txS - txV, dty = tyS - tyV, adtx = fabsf(dtx);
      const float zm = (((p.mag[0] + p.mag[1] * adtx) + p.mag[2] * (dtx * dtx)) + p.mag[3] * fabsf(xS)) +
                       p.mag[4] * (txV * txV);                                     // Eq. 18
      const float xs = xS + (zm - p.zS) * txS, xv = xV + (zm - p.zV) * txV;        // Eq. 17
      const float ys = yS + p.dzyS * tyS, yv = yV + p.dzyV * tyV;
      float in[8];
      in[0] = zm; in[1] = xs - xv; in[2] = ys - yv; in[3] = dtx; in[4] = dty; in[5] = m.chi2;
      in[6] = nn_eta(txV, tyV);
      in[7] = (float)(p.snx && p.snuv ? (int)p.snx[slot] + (int)p.snuv[slot] : 12);
      const float g = nn_ghost_prob(p.nn, in);
      m.ghost = g;
      if (g < nn_cut) {
        atomicMin(&seed_best[s], (unsigned long long)__float_as_uint(g));
        atomicMin(&velo_best[sorig[v]], (unsigned long long)__float_as_uint(g));
      }
    }
    __syncthreads();
  } else {
  for (int k = tid; k < nm; k += kMatchThreads) {
    const MatchCand& m = mc[k];
    if ((m.key >> 50) <= key_ok)
      atomicMin(&seed_best[m.seed], ((unsigned long long)__float_as_uint(m.chi2) << 32) | sorig[m.velo]);
  }
  __syncthreads();
  LHCB_CLK(12)
  // ---- M4: one-to-one selection (O14) -------------------------------------------------------------
  for (int k = tid; k < nm; k += kMatchThreads) {
    const MatchCand& m = mc[k];
    if ((m.key >> 50) > key_ok) continue;
    const unsigned long long cb = (unsigned long long)__float_as_uint(m.chi2) << 32;
    if (seed_best[m.seed] != (cb | sorig[m.velo])) continue;
    atomicMin(&velo_best[sorig[m.velo]], cb | m.seed);
  }
  __syncthreads();
  // Reading A21: an exact chi2 tie between two seeds for one VELO state (twin seeds: bit-identical states
  // from duplicate hits) is decided by the seeds' hit lists, not by their slot order.  Ties are detected by
  // every thread; the (rare) event that has one resolves it serially.
  for (int k = tid; k < nm; k += kMatchThreads) {
    const MatchCand& m = mc[k];
    if ((m.key >> 50) > key_ok) continue;
    const unsigned long long cb = (unsigned long long)__float_as_uint(m.chi2) << 32;
    if (seed_best[m.seed] != (cb | sorig[m.velo])) continue;
    const unsigned long long vb = velo_best[sorig[m.velo]];
    if ((vb >> 32) == (cb >> 32) && (uint32_t)vb != (uint32_t)m.seed) hdr[9] = 1;
  }
  __syncthreads();
  if (hdr[9]) {
    if (tid == 0) {
      auto slot_of = [&](int s) { return s < c0 ? (size_t)(2 * e) * p.max_seeds + s : (size_t)(2 * e + 1) * p.max_seeds + (s - c0); };
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
  for (int k = tid; k < nm; k += kMatchThreads) {
    const MatchCand& m = mc[k];
    if ((m.key >> 50) > key_ok) continue;
    const unsigned long long cb = (unsigned long long)__float_as_uint(m.chi2) << 32;
    const int vo = sorig[m.velo];
    if (use_nn) {
      // kept if below the cut and no track sharing its seed or its VELO is better by the margin (the minimum
      // includes the track itself, which never satisfies g >= g + margin)
      if (!(m.ghost < nn_cut)) continue;
      const float gs = __uint_as_float((unsigned int)seed_best[m.seed]), gv = __uint_as_float((unsigned int)velo_best[vo]);
      if (m.ghost >= gs + nn_margin || m.ghost >= gv + nn_margin) continue;
    } else if (seed_best[m.seed] != (cb | vo) || velo_best[vo] != (cb | m.seed)) continue;
    const int slot = atomicAdd(&hdr[1], 1);
    if (slot >= p.max_long) continue;
    const size_t o = (size_t)e * p.max_long + slot, ct = p.long_cap_total;
    const int s = m.seed;
    p.seed_idx[o] = s < c0 ? (uint32_t)((2 * e) * p.max_seeds + s) : (uint32_t)((2 * e + 1) * p.max_seeds + (s - c0));
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
    if (use_nn && p.ghost) p.ghost[o] = m.ghost;
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
