// Event preparation kernel for sm_100a: raw, unsorted SciFi hits -> the tiled, sorted layout the Seeding
// reads (hits tiled by detector half and layer; the searches of section 3 need them sorted
// in x).  SURVEY.md section 8(f)1.  Result = stable sort by (zone, x, raw index) inside each event.
//
// One CTA per event, everything in shared memory, no comparison network:
//   P1  histogram over 24 zones x 256 x-bins (the bin is monotone in x)         one shared atomic per hit
//   P2  exclusive scan of the 6,144 cells (24 per thread + block scan); the cells at the zone starts are
//       the event's zone offsets
//   P3  scatter (x, raw index, zone) into the cell's range                        one shared atomic per hit
//   P4  thread per scattered hit: its cell from its zone and x; rank inside the cell
//       (about 0.6 hits per cell at nominal occupancy) by the literal comparison (x, raw index) <
//       (x', raw index'); hit_x and perm are written at cell start + rank, i.e. within a few elements of the
//       thread's own position: nearly coalesced stores
// The 6,144 cell counters are 16-bit (an event has at most 65,535 hits), two per 32-bit word, so that four
// 512-thread CTAs fit an SM at the nominal capacity.
// Bins only group; the order is decided by exact float comparisons, so the output is bit-identical to a
// stable sort whatever the rounding of the bin function.
#pragma once
#include <cstdint>

#include "../../include/lhcb.h"
#include "seeding.cuh"   // block_exscan

namespace lhcb {

constexpr int kPrepThreads = 512;
#ifndef LHCB_PREP_BINS
#define LHCB_PREP_BINS 256
#endif
constexpr int kPrepBins = LHCB_PREP_BINS;         // x bins per zone
constexpr int kPrepCells = 24 * kPrepBins;        // 24 cells per thread
static_assert(kPrepCells % kPrepThreads == 0, "whole cells per thread");

struct PrepParams {
  float x_lo, scale;          // bin(x) = clamp((x - x_lo) * scale, 0, kPrepBins - 1)
  int max_hits;               // raw hits of one event that fit in shared memory
  int n_events;
  const uint32_t* raw_off;
  const float* raw_x;
  const uint8_t* raw_zone;
  uint32_t* zone_off;
  float* hit_x;
  uint32_t* perm;             // may be NULL
  uint32_t* status;
};

__host__ __device__ inline size_t prep_smem_bytes(int max_hits) {
  size_t b = (size_t)kPrepCells * 2 + 512;                       // packed cells; scan scratch, zone starts, flag
  b += (((size_t)max_hits * 4 + 15) & ~(size_t)15);              // x by cell
  b += (((size_t)max_hits * 2 + 15) & ~(size_t)15);              // raw index (event-local) by cell
  b += (((size_t)max_hits + 15) & ~(size_t)15);                  // zone by cell
  return b;
}

// 16-bit cell c lives in half (c & 1) of word c >> 1
__device__ __forceinline__ unsigned int cell_add(unsigned int* cw, int c) {
  const int sh = (c & 1) << 4;
  return (atomicAdd(&cw[c >> 1], 1u << sh) >> sh) & 0xFFFFu;
}
__device__ __forceinline__ int cell_get(const unsigned int* cw, int c) {
  return (int)((cw[c >> 1] >> ((c & 1) << 4)) & 0xFFFFu);
}

__device__ __forceinline__ int prep_cell(const PrepParams& p, float x, int zone) {
  float t = (x - p.x_lo) * p.scale;
  t = fminf(fmaxf(t, 0.f), (float)(kPrepBins - 1));
  return zone * kPrepBins + (int)t;
}

__global__ void __launch_bounds__(kPrepThreads)
prepare_kernel(const __grid_constant__ PrepParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  unsigned int* cw = reinterpret_cast<unsigned int*>(smem);                       // kPrepCells / 2 words
  int* warp_sums = reinterpret_cast<int*>(smem + (size_t)kPrepCells * 2);         // [kPrepThreads / 32 + 1]
  int* flag = warp_sums + 72;
  float* sx = reinterpret_cast<float*>(smem + (size_t)kPrepCells * 2 + 512);
  uint16_t* sidx = reinterpret_cast<uint16_t*>(reinterpret_cast<unsigned char*>(sx) +
                                               (((size_t)p.max_hits * 4 + 15) & ~(size_t)15));
  uint8_t* szone = reinterpret_cast<uint8_t*>(sidx) + (((size_t)p.max_hits * 2 + 15) & ~(size_t)15);
  constexpr int T = kPrepThreads, per = kPrepCells / kPrepThreads;
  const int tid = threadIdx.x, e = blockIdx.x;
  const uint32_t b = p.raw_off[e];
  const int n = (int)(p.raw_off[e + 1] - b);
  uint32_t* zo = p.zone_off + (size_t)e * 24;
  if (e == p.n_events - 1 && tid == 0) p.zone_off[(size_t)p.n_events * 24] = b + (uint32_t)n;
  const bool too_many = n > p.max_hits || n > 65535;
  for (int c = tid; c < kPrepCells / 2; c += T) cw[c] = 0u;
  if (tid == 0) *flag = 0;
  __syncthreads();
  // P1
  if (!too_many)
#pragma unroll 4
    for (int i = tid; i < n; i += T) {
      const float x = p.raw_x[b + i];
      const int z = p.raw_zone[b + i];
      if (z >= 24 || !(fabsf(x) <= 3.0e38f)) *flag = 1;          // invalid zone, NaN or infinity
      else cell_add(cw, prep_cell(p, x, z));
    }
  __syncthreads();
  if (too_many || *flag) {
    // the event is passed through unsorted, all of it in zone 0, and reported: never silent
    if (tid < 24) zo[tid] = tid == 0 ? b : b + (uint32_t)n;
    for (int i = tid; i < n; i += T) {
      p.hit_x[b + i] = p.raw_x[b + i];
      if (p.perm) p.perm[b + i] = b + (uint32_t)i;
    }
    if (tid == 0) p.status[e] = too_many ? LHCB_ST_HITS_OVERFLOW : LHCB_ST_BAD_RAW_HIT;
    return;
  }
  // P2
  {
    static_assert(per % 2 == 0, "whole words per thread");
    unsigned int v[per];
    int sum = 0;
#pragma unroll
    for (int k = 0; k < per / 2; ++k) {
      const unsigned int w = cw[tid * (per / 2) + k];
      v[2 * k] = w & 0xFFFFu; v[2 * k + 1] = w >> 16;
      sum += (int)(v[2 * k] + v[2 * k + 1]);
    }
    int total;
    int flip = 0;                                          // a single scan: only the first warp_sums buffer is used
    int run = block_exscan<T>(sum, warp_sums, flip, total);
#pragma unroll
    for (int k = 0; k < per / 2; ++k) {
      const unsigned int lo = (unsigned int)run; run += (int)v[2 * k];
      const unsigned int hi = (unsigned int)run; run += (int)v[2 * k + 1];
      cw[tid * (per / 2) + k] = lo | (hi << 16);
    }
  }
  __syncthreads();
  if (tid < 24) zo[tid] = b + (uint32_t)cell_get(cw, tid * kPrepBins);
  if (tid == 0) p.status[e] = 0u;
  __syncthreads();
  // P3
#pragma unroll 4
  for (int i = tid; i < n; i += T) {
    const float x = p.raw_x[b + i];
    const int z = p.raw_zone[b + i];
    const unsigned int pos = cell_add(cw, prep_cell(p, x, z));
    sx[pos] = x;
    sidx[pos] = (uint16_t)i;
    szone[pos] = (uint8_t)z;
  }
  __syncthreads();
  // P4: the cell counters now hold the end of each cell = the start of the next one
  for (int q = tid; q < n; q += T) {
    const float x = sx[q];
    const int i = sidx[q];
    const int z = szone[q];
    const int c = prep_cell(p, x, z);
    const int start = c ? cell_get(cw, c - 1) : 0, end = cell_get(cw, c);
    int rank = 0;
    for (int r = start; r < end; ++r) {
      const float xr = sx[r];
      rank += (xr < x || (xr == x && (int)sidx[r] < i)) ? 1 : 0;
    }
    const uint32_t out = b + (uint32_t)(start + rank);
    p.hit_x[out] = x;
    if (p.perm) p.perm[out] = b + (uint32_t)i;
  }
}

}  // namespace lhcb
