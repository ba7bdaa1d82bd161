// Event preparation kernel for sm_100a: raw, unsorted SciFi hits -> the tiled, sorted layout the Seeding
// reads (hits tiled by detector half and layer; the searches of section 3 need them sorted
// in x).  SURVEY.md section 8(f)1.  Result = stable sort by (zone, x, raw index) inside each event.
//
// One CTA per event, no comparison network.  Thread t owns the raw hits t, t + T, t + 2T, ... (coalesced
// loads) and keeps one packed register per hit from the first pass to the last, so that every pass after the
// first is a pass over registers, not over memory:
//   P1  histogram over 24 zones x 256 x-bins (the bin is monotone in x): one shared atomic per hit; its return
//       value is the hit's ARRIVAL RANK inside its cell, kept with the cell number
//   P2  exclusive scan of the 6,144 cells (12 per thread + block scan); the cells at the zone starts are the
//       event's zone offsets
//   P3  every hit goes to (start of its cell + arrival rank) in shared memory: no second atomic
//   P4  the cells with more than one member (queued during P2; about 800 of the 6,144 at nominal occupancy)
//       are put in order, one thread per cell, by an insertion sort with the literal comparison (x, raw index)
//       < (x', raw index'); more than half of the hits are alone in their cell and are already in place
//   P5  hit_x and perm leave shared memory with 16-byte stores (the shared arrays are shifted by the event's
//       misalignment so that shared and global addresses are aligned together)
// The 6,144 cell counters are 16-bit (an event has at most 65,535 hits), two per 32-bit word.
// Bins only group; the order is decided by exact float comparisons, so the output is bit-identical to a
// stable sort whatever the rounding of the bin function.  A cell that collects more than kPrepCellMax hits
// (never at any sane occupancy: it takes that many hits within 25 mm in one zone, or outside the binned range)
// sends the event to a plain all-pairs ranking (prep_all_pairs), slow and obviously the same order.
#pragma once
#include <cstdint>

#include "../../include/lhcb.h"
#include "seeding.cuh"   // block_exscan

namespace lhcb {

#ifndef LHCB_PREP_BINS
#define LHCB_PREP_BINS 256
#endif
constexpr int kPrepBins = LHCB_PREP_BINS;         // x bins per zone
constexpr int kPrepCells = 24 * kPrepBins;
#ifndef LHCB_PREP_BATCH
#define LHCB_PREP_BATCH 4
#endif
constexpr int kPrepBatch = LHCB_PREP_BATCH;       // raw hits a thread loads before it processes them
constexpr int kPrepCellMax = 64;                  // members of a cell the one-thread insertion sort handles

struct PrepParams {
  float x_lo, scale;          // bin(x) = clamp((x - x_lo) * scale, 0, kPrepBins - 1)
  int max_hits;               // raw hits of one event that fit in shared memory (and in T * R registers)
  int n_events;
  const uint32_t* raw_off;
  const float* raw_x;
  const uint8_t* raw_zone;
  uint32_t* zone_off;
  float* hit_x;
  uint32_t* perm;             // may be NULL
  uint32_t* status;
};

typedef uint16_t prep_cell_t;                     // 16-bit cells, two per word (an event has at most 65,535 hits): the
                                                  // counters take 12 KB and four 512-thread CTAs share an SM

// [cells | scan scratch, flag, queue length | x by position, shifted by up to 3 | raw index by position,
//  shifted | queue of the cells with more than one member]
__host__ __device__ inline int prep_queue_cap(int max_hits) { return max_hits / 2 < kPrepCells ? max_hits / 2 : kPrepCells; }
__host__ __device__ inline size_t prep_smem_bytes(int max_hits) {
  size_t b = (size_t)kPrepCells * sizeof(prep_cell_t) + 512;
  b += (((size_t)max_hits + 8) * 4 + 15) & ~(size_t)15;
  b += (((size_t)max_hits + 8) * 2 + 15) & ~(size_t)15;
  b += ((size_t)prep_queue_cap(max_hits) * 2 + 15) & ~(size_t)15;
  return b;
}

__device__ __forceinline__ unsigned int cell_inc(unsigned int* cw, int c) {      // returns the count before
  const int sh = (c & 1) << 4;
  return (atomicAdd(&cw[c >> 1], 1u << sh) >> sh) & 0xFFFFu;
}
__device__ __forceinline__ int cell_start(const unsigned int* cw, int c) {
  return (int)((cw[c >> 1] >> ((c & 1) << 4)) & 0xFFFFu);
}

__device__ __forceinline__ int prep_cell(const PrepParams& p, float x, int zone) {
  float t = (x - p.x_lo) * p.scale;
  t = fminf(fmaxf(t, 0.f), (float)(kPrepBins - 1));
  return zone * kPrepBins + (int)t;
}

// The definition written out, for the events the fast passes decline: the position of a hit is the number of
// hits of its event that precede it in (zone, x, raw index) order.  O(n^2) reads of the raw arrays.
template <int T>
__device__ void prep_all_pairs(const PrepParams& p, uint32_t b, int n, uint32_t* zo) {
  const int tid = threadIdx.x;
  for (int i = tid; i < n; i += T) {
    const float x = p.raw_x[b + i];
    const int z = p.raw_zone[b + i];
    int rank = 0;
    for (int j = 0; j < n; ++j) {
      const float xj = p.raw_x[b + j];
      const int zj = p.raw_zone[b + j];
      rank += (zj < z || (zj == z && (xj < x || (xj == x && j < i)))) ? 1 : 0;
    }
    p.hit_x[b + rank] = x;
    if (p.perm) p.perm[b + rank] = b + (uint32_t)i;
  }
  if (tid < 24) {
    int below = 0;
    for (int j = 0; j < n; ++j) below += (int)p.raw_zone[b + j] < tid ? 1 : 0;
    zo[tid] = b + (uint32_t)below;
  }
}

// T threads, R hits per thread: an event of up to T * R hits (>= p.max_hits by the choice of the instantiation)
template <int T, int R, int MIN_CTAS>
__global__ void __launch_bounds__(T, MIN_CTAS)
prepare_kernel(const __grid_constant__ PrepParams p) {
  extern __shared__ __align__(16) unsigned char smem[];
  unsigned int* cw = reinterpret_cast<unsigned int*>(smem);                       // kPrepCells counters, then cell starts
  int* warp_sums = reinterpret_cast<int*>(smem + (size_t)kPrepCells * sizeof(prep_cell_t));         // [2][kSeedThreadsMax / 32 + 1] at most
  int* flag = warp_sums + 100;
  float* sx = reinterpret_cast<float*>(smem + (size_t)kPrepCells * sizeof(prep_cell_t) + 512);
  uint16_t* si = reinterpret_cast<uint16_t*>(reinterpret_cast<unsigned char*>(sx) +
                                             ((((size_t)p.max_hits + 8) * 4 + 15) & ~(size_t)15));
  uint16_t* qcell = si + (((size_t)p.max_hits + 8 + 7) & ~(size_t)7);
  constexpr int per = kPrepCells / T;
  static_assert(per * T == kPrepCells && per % 2 == 0, "whole words of cells per thread");
  static_assert(T <= kSeedThreadsMax * 2, "scan scratch");
  const int tid = threadIdx.x, e = blockIdx.x;
  const uint32_t b = p.raw_off[e];
  const int n = (int)(p.raw_off[e + 1] - b);
  uint32_t* zo = p.zone_off + (size_t)e * 24;
  if (e == p.n_events - 1 && tid == 0) p.zone_off[(size_t)p.n_events * 24] = b + (uint32_t)n;
  const bool too_many = n > p.max_hits || n > 65535 || n > T * R;
  for (int c = tid; c < kPrepCells * (int)sizeof(prep_cell_t) / 16; c += T) reinterpret_cast<uint4*>(cw)[c] = make_uint4(0u, 0u, 0u, 0u);
  if (tid == 0) *flag = 0;
  __syncthreads();
  const float* __restrict__ rx = p.raw_x + b;
  const uint8_t* __restrict__ rz = p.raw_zone + b;
  // ---- P1: cell and arrival rank of every hit -> A[r] = cell | arrival << 16
  uint32_t A[R];
  if (!too_many) {
#pragma unroll
    for (int r0 = 0; r0 < R; r0 += kPrepBatch) {             // kPrepBatch independent loads in flight per thread
      if (r0 * T >= n) {                                     // (uniform) no hits in these rounds
#pragma unroll
        for (int q = 0; q < kPrepBatch; ++q) if (r0 + q < R) A[r0 + q] = 0u;
        continue;
      }
      float x[kPrepBatch];
      int z[kPrepBatch];
#pragma unroll
      for (int q = 0; q < kPrepBatch; ++q) {
        const int i = tid + (r0 + q) * T;
        x[q] = 0.f; z[q] = 0;
        if (r0 + q < R && i < n) { x[q] = __ldg(rx + i); z[q] = __ldg(rz + i); }
      }
#pragma unroll
      for (int q = 0; q < kPrepBatch; ++q) {
        const int i = tid + (r0 + q) * T;
        if (r0 + q < R) {
          A[r0 + q] = 0u;
          if (i < n) {
            if (z[q] >= 24 || !(fabsf(x[q]) <= 3.0e38f)) *flag = 1;          // invalid zone, NaN or infinity
            else {
              const int c = prep_cell(p, x[q], z[q]);
              LHCB_CHECK_IDX(c, kPrepCells);
              const unsigned int arr = cell_inc(cw, c);
              if (arr >= (unsigned)kPrepCellMax) atomicOr(flag, 2);
              A[r0 + q] = (uint32_t)c | (arr << 16);
            }
          }
        }
      }
    }
  }
  __syncthreads();
  const int fl = *flag;
  if (too_many || (fl & 1)) {
    // the event is passed through unsorted, all of it in zone 0, and reported: never silent
    if (tid < 24) zo[tid] = tid == 0 ? b : b + (uint32_t)n;
    for (int i = tid; i < n; i += T) {
      p.hit_x[b + i] = p.raw_x[b + i];
      if (p.perm) p.perm[b + i] = b + (uint32_t)i;
    }
    if (tid == 0) p.status[e] = (n > p.max_hits || n > 65535 || n > T * R) ? LHCB_ST_HITS_OVERFLOW : LHCB_ST_BAD_RAW_HIT;
    return;
  }
  if (fl & 2) {                                              // a cell beyond kPrepCellMax members: the definition, written out
    prep_all_pairs<T>(p, b, n, zo);
    if (tid == 0) p.status[e] = 0u;
    return;
  }
  // ---- P2: exclusive scan of the cells; the cells with more than one member are queued for P4
  int nqueued = 0;
  {
    unsigned int v[per];
    int sum = 0;
    unsigned int mmask = 0u;                                 // my cells with more than one member
#pragma unroll
    for (int k = 0; k < per / 2; ++k) {
      const unsigned int w = cw[tid * (per / 2) + k];
      v[2 * k] = w & 0xFFFFu; v[2 * k + 1] = w >> 16;
    }
#pragma unroll
    for (int k = 0; k < per; ++k) {
      sum += (int)v[k];
      mmask |= (v[k] >= 2u ? 1u : 0u) << k;
    }
    const int multi = __popc(mmask);
    // one scan for both prefix sums: hits in the low half (an event has at most 65,535), queued cells above
    int total;
    int flip = 0;                                            // a single scan: only the first warp_sums buffer is used
    const int ex = block_exscan<T>(sum | (multi << 16), warp_sums, flip, total);
    int run = ex & 0xFFFF, qpos = ex >> 16;
    nqueued = total >> 16;
    while (mmask) {
      LHCB_CHECK_IDX(qpos, prep_queue_cap(p.max_hits));
      qcell[qpos++] = (uint16_t)(tid * per + __ffs(mmask) - 1);
      mmask &= mmask - 1u;
    }
#pragma unroll
    for (int k = 0; k < per / 2; ++k) {
      const unsigned int lo = (unsigned int)run; run += (int)v[2 * k];
      const unsigned int hi = (unsigned int)run; run += (int)v[2 * k + 1];
      cw[tid * (per / 2) + k] = lo | (hi << 16);
    }
  }
  __syncthreads();
  if (tid < 24) zo[tid] = b + (uint32_t)cell_start(cw, tid * kPrepBins);
  if (tid == 0) p.status[e] = 0u;
  // ---- P3: every hit to (start of its cell + arrival rank).
  // Position q of the event lives at index q + sh of the shared arrays, sh = b mod 4: shared and global
  // addresses are then 16-byte aligned together (P5).
  const int sh = (int)(b & 3u);
#pragma unroll
  for (int r0 = 0; r0 < R; r0 += 4) {
    if (r0 * T >= n) continue;
    float x[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int i = tid + (r0 + q) * T;
      x[q] = 0.f;
      if (r0 + q < R && i < n) x[q] = __ldg(rx + i);         // second read: served by L2
    }
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int i = tid + (r0 + q) * T;
      if (r0 + q < R && i < n) {
        const uint32_t a = A[r0 + q];
        const int dst = sh + cell_start(cw, (int)(a & 0xFFFFu)) + (int)(a >> 16);
        LHCB_CHECK_IDX(dst - sh, n);
        sx[dst] = x[q];
        si[dst] = (uint16_t)i;
      }
    }
  }
  __syncthreads();
  // ---- P4: order inside the queued cells (more than one member), one thread per cell
  {
    for (int q = tid; q < nqueued; q += T) {
      const int c = qcell[q];
      const int start = cell_start(cw, c), cnt = (c + 1 < kPrepCells ? cell_start(cw, c + 1) : n) - start;
      LHCB_CHECK_IDX(start + cnt, n + 1); LHCB_CHECK_IDX(cnt - 2, kPrepCellMax);
      float* cx = sx + sh + start;
      uint16_t* ci = si + sh + start;
      for (int a = 1; a < cnt; ++a) {
        const float xa = cx[a];
        const uint16_t ia = ci[a];
        int m = a;
        while (m > 0) {
          const float xm = cx[m - 1];
          const uint16_t im = ci[m - 1];
          if (xm < xa || (xm == xa && im < ia)) break;
          cx[m] = xm; ci[m] = im;
          --m;
        }
        cx[m] = xa; ci[m] = ia;
      }
    }
  }
  __syncthreads();
  // ---- P5: out with 16-byte stores where hit_x / perm are 16-byte aligned (cudaMalloc'ed arrays are)
  const bool vec = ((reinterpret_cast<uintptr_t>(p.hit_x) | (p.perm ? reinterpret_cast<uintptr_t>(p.perm) : 0)) & 15) == 0;
  if (vec) {
    float* __restrict__ gx = p.hit_x + (b - (uint32_t)sh);
    uint32_t* __restrict__ gp = p.perm ? p.perm + (b - (uint32_t)sh) : nullptr;
    const int nv = (n + sh + 3) >> 2;
    for (int v = tid; v < nv; v += T) {
      const int q = 4 * v;
      const float4 xv = *reinterpret_cast<const float4*>(sx + q);
      const uint2 iv = *reinterpret_cast<const uint2*>(si + q);
      const uint4 pv = make_uint4(b + (iv.x & 0xFFFFu), b + (iv.x >> 16), b + (iv.y & 0xFFFFu), b + (iv.y >> 16));
      if (q >= sh && q + 3 < n + sh) {
        *reinterpret_cast<float4*>(gx + q) = xv;
        if (gp) *reinterpret_cast<uint4*>(gp + q) = pv;
      } else {                                               // the first and the last vector of the event
        const float xs[4] = {xv.x, xv.y, xv.z, xv.w};
        const uint32_t ps[4] = {pv.x, pv.y, pv.z, pv.w};
#pragma unroll
        for (int k = 0; k < 4; ++k)
          if (q + k >= sh && q + k < n + sh) {
            gx[q + k] = xs[k];
            if (gp) gp[q + k] = ps[k];
          }
      }
    }
  } else {
    for (int q = tid; q < n; q += T) {
      p.hit_x[b + q] = sx[sh + q];
      if (p.perm) p.perm[b + q] = b + (uint32_t)si[sh + q];
    }
  }
}

}  // namespace lhcb
