// Scheduling and output compaction kernels around the two hot kernels (PAPER.md L384:
// batches of about 1000 events).
//
//   order_kernel    heaviest first: the event-halves (Seeding) and the events (Matching) of a batch are
//                   bucket-sorted by their number of SciFi / UT hits, descending.  A batch of 1,024 events is
//                   only 3.5 waves of Seeding CTAs on 148 SMs; started in this order the short CTAs fill the
//                   last wave.  The order only permutes CTAs: every output stays in the slots of its own
//                   event(-half).
//   compact_scan    exclusive prefix of the per-half seed counts and of the per-event long-track counts of a
//                   slice, continued from the running totals of the previous slice
//   compact_gather  seeds and long tracks from their fixed slots to dense arrays (what the host-buffer
//                   pipeline copies back); the seed reference of a long track becomes an index into the dense
//                   seed arrays
#pragma once
#include <cstdint>

#include "../../include/lhcb.h"

namespace lhcb {

constexpr int kOrderThreads = 1024;
constexpr int kOrderBuckets = 256;

// weight -> bucket, heaviest first
__device__ __forceinline__ int order_bucket(uint32_t w, int shift) {
  const uint32_t b = w >> shift;
  return kOrderBuckets - 1 - (int)(b < (uint32_t)kOrderBuckets ? b : (uint32_t)kOrderBuckets - 1);
}

constexpr int kOrderPerThread = 32;   // weights a thread keeps in registers between the two passes
#ifndef LHCB_ORDER_MAX_SORTED
#define LHCB_ORDER_MAX_SORTED 3072
#endif
constexpr int kOrderMaxSorted = LHCB_ORDER_MAX_SORTED; // batches above this many events run without the workspace (host decision, lhcb_api.cu)

// one CTA.  seed_order[2 n_events], match_order[n_events] (either may be NULL), done[2 n_events].  Without UT
// offsets and without VELO offsets there is nothing to weigh the events by: match_order is then the identity, so
// that a workspace this kernel has filled is valid for lhcb_matching whatever lhcb_order was given.
// Up to 32 halves per thread (32,768 halves: the 16,384-event batch) are loaded once, all loads in flight
// together, and kept in registers for the scatter pass; larger batches take a plain two-pass loop.
__global__ void __launch_bounds__(kOrderThreads)
order_kernel(int n_events, const uint32_t* __restrict__ zone_off, const uint32_t* __restrict__ ut_off,
             const uint32_t* __restrict__ velo_off, uint32_t* __restrict__ seed_order, uint32_t* __restrict__ match_order,
             uint32_t* __restrict__ done) {
  __shared__ int cur[2][kOrderBuckets];
  const int tid = threadIdx.x;
  for (int i = tid; i < 2 * kOrderBuckets; i += kOrderThreads) (&cur[0][0])[i] = 0;
  const int nh = 2 * n_events;
  // "seeds are in global memory" flags: up unless a Seeding run lowers them (a Matching on given seeds passes)
  for (int h = tid; h < nh; h += kOrderThreads) done[h] = 1u;
  const bool fast = nh <= kOrderThreads * kOrderPerThread;
  if (match_order && !ut_off && !velo_off) {
    for (int e = tid; e < n_events; e += kOrderThreads) match_order[e] = (uint32_t)e;
    match_order = nullptr;                                  // nothing to sort
  }
  auto seed_w = [&](int h) { return zone_off[(size_t)h * 12 + 12] - zone_off[(size_t)h * 12]; };
  auto match_w = [&](int e) {
    return ut_off ? ut_off[(size_t)e * 4 + 4] - ut_off[(size_t)e * 4] : 32u * (velo_off[e + 1] - velo_off[e]);
  };
  uint8_t bs[kOrderPerThread], bm[kOrderPerThread / 2];
  if (fast) {
#pragma unroll
    for (int k = 0; k < kOrderPerThread; ++k) {
      const int h = tid + k * kOrderThreads;
      bs[k] = (seed_order && h < nh) ? (uint8_t)order_bucket(seed_w(h), 4) : (uint8_t)0;
    }
#pragma unroll
    for (int k = 0; k < kOrderPerThread / 2; ++k) {
      const int e = tid + k * kOrderThreads;
      bm[k] = (match_order && e < n_events) ? (uint8_t)order_bucket(match_w(e), 5) : (uint8_t)0;
    }
  }
  __syncthreads();
  if (fast) {
#pragma unroll
    for (int k = 0; k < kOrderPerThread; ++k)
      if (seed_order && tid + k * kOrderThreads < nh) atomicAdd(&cur[0][bs[k]], 1);
#pragma unroll
    for (int k = 0; k < kOrderPerThread / 2; ++k)
      if (match_order && tid + k * kOrderThreads < n_events) atomicAdd(&cur[1][bm[k]], 1);
  } else {
    if (seed_order)
      for (int h = tid; h < nh; h += kOrderThreads) atomicAdd(&cur[0][order_bucket(seed_w(h), 4)], 1);
    if (match_order)
      for (int e = tid; e < n_events; e += kOrderThreads) atomicAdd(&cur[1][order_bucket(match_w(e), 5)], 1);
  }
  __syncthreads();
  if (tid < 64) {                                           // exclusive scan of the 256 buckets of each list, one warp each
    const int which = tid >> 5, lane = tid & 31;
    int run = 0;
    for (int c = 0; c < kOrderBuckets / 32; ++c) {
      const int v = cur[which][c * 32 + lane];
      int inc = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
      }
      cur[which][c * 32 + lane] = run + inc - v;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
  }
  __syncthreads();
  if (fast) {
#pragma unroll
    for (int k = 0; k < kOrderPerThread; ++k) {
      const int h = tid + k * kOrderThreads;
      if (seed_order && h < nh) seed_order[atomicAdd(&cur[0][bs[k]], 1)] = (uint32_t)h;
    }
#pragma unroll
    for (int k = 0; k < kOrderPerThread / 2; ++k) {
      const int e = tid + k * kOrderThreads;
      if (match_order && e < n_events) match_order[atomicAdd(&cur[1][bm[k]], 1)] = (uint32_t)e;
    }
  } else {
    if (seed_order)
      for (int h = tid; h < nh; h += kOrderThreads) seed_order[atomicAdd(&cur[0][order_bucket(seed_w(h), 4)], 1)] = (uint32_t)h;
    if (match_order)
      for (int e = tid; e < n_events; e += kOrderThreads) match_order[atomicAdd(&cur[1][order_bucket(match_w(e), 5)], 1)] = (uint32_t)e;
  }
}

// UT strip numbers -> x0 for the hits [range[0], range[1]) (read on the device: the grid is fixed, so the
// launch can sit in a CUDA graph).  x0 = x_origin + strip * pitch, two float32 operations (-fmad=false).
__global__ void ut_decode_kernel(const uint32_t* __restrict__ range_begin, const uint32_t* __restrict__ range_end,
                                 const uint16_t* __restrict__ strip, float* __restrict__ x0, float x_origin, float pitch) {
  const uint32_t b = *range_begin, e = *range_end;
  for (uint32_t i = b + blockIdx.x * blockDim.x + threadIdx.x; i < e; i += gridDim.x * blockDim.x)
    x0[i] = x_origin + (float)strip[i] * pitch;
}

// ---------------------------------------------------------------------------------------------- compaction
struct CompactParams {
  int n_events;                 // events of this slice
  int max_seeds, max_long;      // slots per half / per event
  // slot arrays of the slice (lhcb_seeds_t / lhcb_long_t layout, cap_total = n_events * 2 * max_seeds etc.)
  const uint32_t* s_count; const float* s_state; const float* s_par; const uint32_t* s_hits;
  const uint8_t *s_nx, *s_nuv;
  const uint32_t* l_count; const uint32_t *l_seed, *l_velo, *l_ut; const uint8_t* l_nut;
  const float *l_qop, *l_chi2, *l_ghost;
  // dense arrays of the whole batch (row stride cap_s / cap_l) and their offset tables
  uint32_t* totals;             // [2] running totals {seeds, long tracks} of the batch so far (device)
  uint32_t* slice_totals;       // [4] {seed base, seed end, long base, long end} of this slice, for the host
  uint32_t* s_off;              // [2 n_events + 1] of this slice, absolute (batch) positions
  uint32_t* l_off;              // [n_events + 1]
  uint32_t cap_s, cap_l;
  float* d_state; float* d_par; uint16_t* d_hits; uint8_t *d_nx, *d_nuv;
  const uint32_t* zone_off;     // of this slice: dense hits are zone-local (hit index - first hit of its (half, layer) zone)
  uint32_t *d_seed, *d_velo, *d_ut; uint8_t* d_nut; float *d_qop, *d_chi2, *d_ghost;
  uint32_t long_velo_rebase, long_ut_rebase;   // (reserved: indices are already batch-global)
};

constexpr int kScanThreads = 1024;

// two CTAs: block 0 scans the seed counts (per half), block 1 the long-track counts (per event)
__global__ void __launch_bounds__(kScanThreads)
compact_scan_kernel(const __grid_constant__ CompactParams p) {
  __shared__ uint32_t wsum[kScanThreads / 32];
  __shared__ uint32_t base_s;
  const int which = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = which == 0 ? 2 * p.n_events : p.n_events;
  const uint32_t* cnt = which == 0 ? p.s_count : p.l_count;
  const uint32_t cap = which == 0 ? (uint32_t)p.max_seeds : (uint32_t)p.max_long;
  uint32_t* off = which == 0 ? p.s_off : p.l_off;
  if (tid == 0) base_s = p.totals[which];
  const int per = (n + kScanThreads - 1) / kScanThreads;
  const int i0 = tid * per, i1 = i0 + per < n ? i0 + per : n;
  uint32_t sum = 0;
  for (int i = i0; i < i1; ++i) { const uint32_t c = cnt[i]; sum += c < cap ? c : cap; }
  uint32_t inc = sum;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint32_t w = wsum[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, w, o);
      if (lane >= o) w += t;
    }
    wsum[lane] = w;
  }
  __syncthreads();
  uint32_t run = base_s + (warp ? wsum[warp - 1] : 0u) + inc - sum;
  for (int i = i0; i < i1; ++i) { off[i] = run; const uint32_t c = cnt[i]; run += c < cap ? c : cap; }
  if (tid == kScanThreads - 1) {
    const uint32_t end = base_s + wsum[kScanThreads / 32 - 1];
    off[n] = end;
    p.slice_totals[2 * which] = base_s;
    p.slice_totals[2 * which + 1] = end;
    p.totals[which] = end;
  }
}

constexpr int kGatherThreads = 256;

// warp per group: groups [0, 2 n_events) are event-halves (seeds), the rest events (long tracks)
__global__ void __launch_bounds__(kGatherThreads)
compact_gather_kernel(const __grid_constant__ CompactParams p) {
  const int g = blockIdx.x * (kGatherThreads / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  const int nh = 2 * p.n_events;
  if (g < nh) {
    const uint32_t b = p.s_off[g], n = p.s_off[g + 1] - b;
    if (b + n > p.cap_s) return;                            // dense arrays full: reported by the host from the totals
    const size_t ct = (size_t)nh * p.max_seeds, s0 = (size_t)g * p.max_seeds;
    for (uint32_t i = lane; i < n; i += 32) {
#pragma unroll
      for (int k = 0; k < 5; ++k) p.d_state[(size_t)k * p.cap_s + b + i] = p.s_state[(size_t)k * ct + s0 + i];
#pragma unroll
      for (int k = 0; k < 12; ++k) {
        const uint32_t hg = p.s_hits[(size_t)k * ct + s0 + i];
        p.d_hits[(size_t)k * p.cap_s + b + i] = hg == LHCB_NO_HIT ? (uint16_t)0xFFFF : (uint16_t)(hg - p.zone_off[(size_t)g * 12 + k]);
      }
      if (p.d_par)
#pragma unroll
        for (int k = 0; k < 7; ++k) p.d_par[(size_t)k * p.cap_s + b + i] = p.s_par[(size_t)k * ct + s0 + i];
      p.d_nx[b + i] = p.s_nx[s0 + i];
      p.d_nuv[b + i] = p.s_nuv[s0 + i];
    }
  } else if (g < nh + p.n_events) {
    const int e = g - nh;
    const uint32_t b = p.l_off[e], n = p.l_off[e + 1] - b;
    if (b + n > p.cap_l) return;
    const size_t ct = (size_t)p.n_events * p.max_long, s0 = (size_t)e * p.max_long;
    for (uint32_t i = lane; i < n; i += 32) {
      const uint32_t slot = p.l_seed[s0 + i];               // slot in the slice's seed arrays -> dense index
      const uint32_t half = slot / (uint32_t)p.max_seeds;
      p.d_seed[b + i] = p.s_off[half] + (slot - half * (uint32_t)p.max_seeds);
      p.d_velo[b + i] = p.l_velo[s0 + i];
#pragma unroll
      for (int k = 0; k < 4; ++k) p.d_ut[(size_t)k * p.cap_l + b + i] = p.l_ut[(size_t)k * ct + s0 + i];
      p.d_nut[b + i] = p.l_nut[s0 + i];
      p.d_qop[b + i] = p.l_qop[s0 + i];
      p.d_chi2[b + i] = p.l_chi2[s0 + i];
      if (p.d_ghost && p.l_ghost) p.d_ghost[b + i] = p.l_ghost[s0 + i];
    }
  }
}

}  // namespace lhcb
