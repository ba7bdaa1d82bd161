// C-ABI entry points (include/lhcb.h): argument checks, constant derivation, kernel launches.
// No torch types: plain pointers and sizes.  Built with
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false -shared -Xcompiler -fPIC
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>

#include "../../include/lhcb.h"
#include "derive.h"
#include "matching.cuh"
#include "prepare.cuh"
#include "seeding.cuh"

#ifndef LHCB_SEED_CTAS
#define LHCB_SEED_CTAS 4   // CTAs per SM the 256-thread seeding kernel is compiled for (64 registers per thread)
#endif

struct lhcb_ctx {
  lhcb_geom_t geom;
  lhcb_derived_t der;
  int device;
  float* d_P;
  float* d_Q;
  float* d_nn;        // ghost-killing network on the device
  int nn_on;
  int uv_hough;       // Hough-cluster UV seeding instead of the iterative one
  size_t seed_smem, match_smem, prep_smem;
  int match_threads;  // 128 when six CTAs fit an SM, else 256
  int seed_threads;   // 256 when four CTAs fit the SM's shared memory, else 512
  int seed_ctas;      // CTAs per SM the seeding kernel is compiled for (register budget)
  int last_cuda_error;
  int last_launches;
};

namespace {

int cuda_fail(lhcb_ctx* ctx, cudaError_t e) {
  if (ctx) ctx->last_cuda_error = (int)e;
  return LHCB_ERR_CUDA;
}

#define LHCB_CUDA(ctx, call)                                   \
  do {                                                         \
    cudaError_t err__ = (call);                                \
    if (err__ != cudaSuccess) return cuda_fail((ctx), err__);  \
  } while (0)

template <class T, size_t N>
void copy_arr(T (&dst)[N], const T (&src)[N]) { std::memcpy(dst, src, sizeof(T) * N); }

void fill_seed_params(const lhcb_ctx* c, lhcb::SeedParams& p) {
  const lhcb_derived_t& D = c->der;
  const lhcb_geom_t& g = c->geom;
  std::memset(&p, 0, sizeof(p));
  copy_arr(p.zb, D.zb); copy_arr(p.gz, D.gz); copy_arr(p.tan_a, D.tan_a); copy_arr(p.inv_tan, D.inv_tan);
  copy_arr(p.inv_z, D.inv_z); copy_arr(p.zt, D.zt);
  std::memcpy(p.ywin_a, D.ywin_a, sizeof(p.ywin_a)); std::memcpy(p.ywin_b, D.ywin_b, sizeof(p.ywin_b));
  for (int i = 0; i < 6; ++i) { p.xl[i] = D.xl[i]; p.ul[i] = D.ul[i]; }
  for (int i = 0; i < 12; ++i) p.slot_of_layer[i] = D.slot_of_layer[i];
  for (int i = 0; i < 2; ++i) {
    p.l1[i] = D.l1[i]; p.l2[i] = D.l2[i]; p.l3[i] = D.l3[i];
    p.dx3max[i] = D.dx3max[i]; p.r13[i] = D.r13[i]; p.inv_dz13[i] = D.inv_dz13[i]; p.z1[i] = D.z1[i];
    p.dz12[i] = D.dz12[i]; p.K[i] = D.K[i]; p.inv_K[i] = D.inv_K[i]; p.G13[i] = D.G13[i];
    p.uv_first[i] = g.uv_first_layer[i];
  }
  p.a = D.a; p.b = D.b; p.kappa = D.kappa; p.inv_kappa = D.inv_kappa;
  p.f_lo = D.f_lo; p.f_hi = D.f_hi; p.d_lo = D.d_lo; p.d_hi = D.d_hi;
  p.tol_x = D.tol_x; p.tol_uv = D.tol_uv; p.chi2x_max = D.chi2x_max; p.chi2y_max = D.chi2y_max;
  copy_arr(p.wx, D.wx); copy_arr(p.wy, D.wy);
  p.zbS = D.zbS; p.gS = D.gS; p.gpS = D.gpS;
  p.min_x_hits = g.min_x_hits; p.min_uv_hits = g.min_uv_hits; p.polarity = g.polarity;
  p.max_seeds = g.max_seeds_per_half; p.max_cand = g.max_xz_cand_per_half; p.max_hits = g.max_hits_per_half;
  p.max_trip = g.max_triplets_per_half;
  for (int it = 0; it < 2; ++it) {                         // the three x-layers an iteration extends to, slots of all six
    const int seedl[3] = {D.l1[it], D.l2[it], D.l3[it]};
    int n = 0;
    for (int s = 0; s < 6; ++s) {
      const int l = D.xl[s];
      if (l != seedl[0] && l != seedl[1] && l != seedl[2] && n < 3) { p.ol[it][n] = l; p.os[it][n] = s; ++n; }
    }
    for (int k = 0; k < 3; ++k) p.ss[it][k] = D.slot_of_layer[seedl[k]];
  }
  p.P = c->d_P; p.Q = c->d_Q;
  // Hough-cluster UV seeding (reading A20): 64 t_y = y / z bins per half over the stereo layers, in double
  // from the float geometry, rounded once
  {
    const double zmin = (double)g.scifi_z[D.ul[0]], tol = std::fabs((double)g.y_half_tol);
    const double range = ((double)g.y_max + tol) / zmin;       // the lower half spans [y_min, tol]: the same width when
                                                               // y_min = -y_max; wider halves land in the edge bins
    p.uv_hough = c->uv_hough;
    p.h_tlo[0] = (float)(-tol / zmin); p.h_tlo[1] = (float)((double)g.y_min / zmin);
    p.h_w = (float)(range / 64.0); p.h_invw = (float)(64.0 / range);
  }
}

void fill_match_params(const lhcb_ctx* c, lhcb::MatchParams& p) {
  const lhcb_derived_t& D = c->der;
  const lhcb_geom_t& g = c->geom;
  std::memset(&p, 0, sizeof(p));
  p.zS = D.zS; p.zV = D.zV; p.dzyS = D.dzyS; p.dzyV = D.dzyV;
  copy_arr(p.mag, D.mag); copy_arr(p.presel, D.presel);
  p.cx0 = D.cx0; p.cx1 = D.cx1; p.cy0 = D.cy0; p.cy1 = D.cy1;
  p.inv_tol_tx = D.inv_tol_tx; p.inv_tol_ty = D.inv_tol_ty; p.chi2m_max = D.chi2m_max;
  p.inv_KB = D.inv_KB; p.Ag = D.Ag; p.Bg = D.Bg; p.inv_Bg = D.inv_Bg;
  copy_arr(p.ut_dz, D.ut_dz); copy_arr(p.ut_dz2, D.ut_dz2); copy_arr(p.ut_dz4, D.ut_dz4);
  copy_arr(p.ut_tan, D.ut_tan); p.ut_y_tol = D.ut_y_tol;
  p.row_y0 = g.ut_row_y0; p.row_pitch = g.ut_row_pitch;
  std::memcpy(p.ut_loose, D.ut_loose, sizeof(p.ut_loose)); std::memcpy(p.ut_tight, D.ut_tight, sizeof(p.ut_tight));
  p.min_ut_hits = g.min_ut_hits; p.polarity = g.polarity;
  p.max_seeds = g.max_seeds_per_half; p.max_long = g.max_long_per_event;
  p.max_mc = g.max_match_cand_per_event; p.max_velo = g.max_velo_per_event; p.max_ut = g.max_ut_per_event;
}

}  // namespace

extern "C" {

int lhcb_geom_derive(const lhcb_geom_t* g, lhcb_derived_t* out) {
  if (!g || !out) return LHCB_ERR_BAD_ARGUMENT;
  return lhcb::derive(*g, *out);
}

int lhcb_geom_init(const lhcb_geom_t* g, int device, lhcb_ctx** out) {
  if (!g || !out || device < 0) return LHCB_ERR_BAD_ARGUMENT;
  *out = nullptr;
  lhcb_ctx* c = new (std::nothrow) lhcb_ctx();
  if (!c) return LHCB_ERR_BAD_ARGUMENT;
  std::memset(c, 0, sizeof(*c));
  c->geom = *g;
  lhcb::resolve_defaults(c->geom);
  c->device = device;
  const lhcb_geom_t& G = c->geom;
  int rc = lhcb::derive(G, c->der);
  if (rc != LHCB_OK) { delete c; return rc; }
  if (G.max_hits_per_half > 8000 || G.max_xz_cand_per_half > 65535 || G.max_seeds_per_half > 32767 ||
      G.max_velo_per_event > 65535 || G.max_ut_per_event > 65534 || G.max_match_cand_per_event > 16383 || G.max_triplets_per_half < G.max_xz_cand_per_half ||
      (size_t)G.max_triplets_per_half * 8 + (size_t)G.max_xz_cand_per_half * 32 < ((size_t)G.max_hits_per_half + 8) * 4 /* staging buffer */) { delete c; return LHCB_ERR_BAD_ARGUMENT; }
  // 256-thread CTAs, four per SM, when their shared memory fits (228 KB per SM, 1 KB reserved per
  // CTA); else 512-thread CTAs, two (or one) per SM
  c->seed_threads = 256;
  c->seed_smem = lhcb::seed_smem_bytes(G.max_hits_per_half, G.max_xz_cand_per_half, G.max_triplets_per_half);
  c->seed_ctas = LHCB_SEED_CTAS;
  if (c->seed_smem > (size_t)(228 * 1024 / LHCB_SEED_CTAS - 1024)) { c->seed_threads = 512; c->seed_ctas = 2; }
  c->match_threads = 128;
  c->match_smem = lhcb::match_smem_bytes(128, G.max_seeds_per_half, G.max_match_cand_per_event, G.max_velo_per_event,
                                         G.max_ut_per_event);
  if (c->match_smem > (size_t)(228 * 1024 / 6 - 1024)) {
    c->match_threads = 256;
    c->match_smem = lhcb::match_smem_bytes(256, G.max_seeds_per_half, G.max_match_cand_per_event, G.max_velo_per_event,
                                           G.max_ut_per_event);
  }
  c->prep_smem = lhcb::prep_smem_bytes(2 * G.max_hits_per_half);
  cudaError_t e = cudaSetDevice(device);
  int max_optin = 0;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&max_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
  if (e != cudaSuccess) { c->last_cuda_error = (int)e; delete c; return LHCB_ERR_CUDA; }
  if (c->seed_smem > (size_t)max_optin || c->match_smem > (size_t)max_optin || c->prep_smem > (size_t)max_optin) { delete c; return LHCB_ERR_CAPACITY; }
  {
    const void* fn = c->seed_ctas == LHCB_SEED_CTAS ? (const void*)lhcb::seeding_kernel<256, LHCB_SEED_CTAS>
                                       : (const void*)lhcb::seeding_kernel<512, 2>;
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->seed_smem);
  }
  if (e == cudaSuccess)
    e = c->match_threads == 128
            ? cudaFuncSetAttribute(lhcb::matching_kernel<128, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->match_smem)
            : cudaFuncSetAttribute(lhcb::matching_kernel<256, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->match_smem);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(lhcb::prepare_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->prep_smem);
  if (e == cudaSuccess) e = cudaMalloc(&c->d_P, sizeof(c->der.P));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_Q, sizeof(c->der.Q));
  if (e == cudaSuccess) e = cudaMalloc(&c->d_nn, LHCB_GHOST_NN_SIZE * sizeof(float));
  if (e == cudaSuccess) e = cudaMemcpy(c->d_P, c->der.P, sizeof(c->der.P), cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy(c->d_Q, c->der.Q, sizeof(c->der.Q), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(c->d_P); cudaFree(c->d_Q); cudaFree(c->d_nn);
    delete c;
    return LHCB_ERR_CUDA;
  }
  *out = c;
  return LHCB_OK;
}

void lhcb_destroy(lhcb_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  cudaFree(c->d_P);
  cudaFree(c->d_Q);
  cudaFree(c->d_nn);
  delete c;
}

int lhcb_get_geom(const lhcb_ctx* c, lhcb_geom_t* out) {
  if (!c || !out) return LHCB_ERR_BAD_ARGUMENT;
  *out = c->geom;
  return LHCB_OK;
}

size_t lhcb_workspace_bytes(const lhcb_ctx* c, int n_events, size_t n_scifi_hits) {
  (void)c; (void)n_events; (void)n_scifi_hits;
  return 0;   // every intermediate lives in shared memory
}

int lhcb_set_uv_hough(lhcb_ctx* c, int on) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  c->uv_hough = on ? 1 : 0;
  return LHCB_OK;
}

int lhcb_set_ghost_nn(lhcb_ctx* c, const float* nn) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!nn) { c->nn_on = 0; return LHCB_OK; }
  if (!(nn[LHCB_GHOST_NN_SIZE - 1] > 0.0f)) return LHCB_ERR_BAD_ARGUMENT;     // margin must be positive
  LHCB_CUDA(c, cudaSetDevice(c->device));
  LHCB_CUDA(c, cudaMemcpy(c->d_nn, nn, LHCB_GHOST_NN_SIZE * sizeof(float), cudaMemcpyHostToDevice));
  c->nn_on = 1;
  return LHCB_OK;
}

int lhcb_prepare(lhcb_ctx* c, const lhcb_raw_t* raw, uint32_t* zone_off, float* hit_x, uint32_t* perm,
                 uint32_t* status, void* stream) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!raw || raw->n_events < 0 || !zone_off) return LHCB_ERR_BAD_ARGUMENT;
  c->last_launches = 0;
  if (raw->n_events == 0) return LHCB_OK;                    // zone_off[0] is then the caller's to set
  if (!raw->off || !status || (raw->n_hits && (!raw->x || !raw->zone || !hit_x))) return LHCB_ERR_BAD_ARGUMENT;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  lhcb::PrepParams p;
  // bins span +-3.2 m (the SciFi acceptance is |x| < 3 m, BASELINE.json configs[1]); x outside lands in
  // the first or last bin, which costs time, not correctness
  p.x_lo = -3200.0f; p.scale = (float)lhcb::kPrepBins / 6400.0f;
  p.max_hits = 2 * c->geom.max_hits_per_half;
  p.n_events = raw->n_events;
  p.raw_off = raw->off; p.raw_x = raw->x; p.raw_zone = raw->zone;
  p.zone_off = zone_off; p.hit_x = hit_x; p.perm = perm; p.status = status;
  lhcb::prepare_kernel<<<raw->n_events, lhcb::kPrepThreads, c->prep_smem, (cudaStream_t)stream>>>(p);
  LHCB_CUDA(c, cudaGetLastError());
  c->last_launches = 1;
  return LHCB_OK;
}

int lhcb_seeding(lhcb_ctx* c, const lhcb_events_t* ev, lhcb_seeds_t* out, void* workspace, void* stream) {
  (void)workspace;
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!ev || !out || ev->n_events < 0) return LHCB_ERR_BAD_ARGUMENT;
  c->last_launches = 0;
  if (ev->n_events == 0) return LHCB_OK;
  if (!ev->zone_off || (!ev->hit_x && ev->n_hits) || !out->count || !out->state || !out->par || !out->hits ||
      !out->nx || !out->nuv || !out->status)
    return LHCB_ERR_BAD_ARGUMENT;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  lhcb::SeedParams p;
  fill_seed_params(c, p);
  p.n_events = ev->n_events; p.n_hits = ev->n_hits; p.zone_off = ev->zone_off; p.hit_x = ev->hit_x;
  p.pol = ev->polarity;
  p.count = out->count; p.state = out->state; p.par = out->par; p.hits = out->hits; p.nx = out->nx;
  p.nuv = out->nuv; p.status = out->status;
  p.cap_total = (size_t)ev->n_events * 2 * (size_t)c->geom.max_seeds_per_half;
  p.smem_total = (int)c->seed_smem;
  if (c->seed_ctas == LHCB_SEED_CTAS)
    lhcb::seeding_kernel<256, LHCB_SEED_CTAS><<<ev->n_events * 2, 256, c->seed_smem, (cudaStream_t)stream>>>(p);
  else
    lhcb::seeding_kernel<512, 2><<<ev->n_events * 2, 512, c->seed_smem, (cudaStream_t)stream>>>(p);
  LHCB_CUDA(c, cudaGetLastError());
  c->last_launches = 1;
  return LHCB_OK;
}

int lhcb_matching(lhcb_ctx* c, const lhcb_seeds_t* seeds, const lhcb_velo_t* velo, const lhcb_ut_t* ut,
                  lhcb_long_t* out, void* workspace, void* stream) {
  (void)workspace;
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!seeds || !velo || !out || velo->n_events < 0 || seeds->n_events != velo->n_events)
    return LHCB_ERR_BAD_ARGUMENT;
  c->last_launches = 0;
  if (velo->n_events == 0) return LHCB_OK;
  if (!seeds->count || !seeds->state || !velo->off || !out->count || !out->seed_idx || !out->velo_idx ||
      !out->ut_idx || !out->n_ut || !out->qop || !out->chi2 || !out->status)
    return LHCB_ERR_BAD_ARGUMENT;
  if (ut && (!ut->off || !ut->x0 || (!ut->row && (!ut->y_lo || !ut->y_hi)))) return LHCB_ERR_BAD_ARGUMENT;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  lhcb::MatchParams p;
  fill_match_params(c, p);
  p.use_ut = (c->geom.ut_enabled && ut) ? 1 : 0;
  p.n_events = velo->n_events;
  p.seed_count = seeds->count; p.state = seeds->state;
  p.seed_cap_total = (size_t)velo->n_events * 2 * (size_t)c->geom.max_seeds_per_half;
  p.velo_off = velo->off; p.vx = velo->x; p.vy = velo->y; p.vtx = velo->tx; p.vty = velo->ty; p.pol = velo->polarity;
  if (ut) { p.ut_off = ut->off; p.ux = ut->x0; p.uylo = ut->y_lo; p.uyhi = ut->y_hi; p.urow = ut->row; p.n_ut_total = ut->n_hits; }
  p.count = out->count; p.seed_idx = out->seed_idx; p.velo_idx = out->velo_idx; p.ut_idx = out->ut_idx;
  p.n_ut = out->n_ut; p.qop = out->qop; p.chi2 = out->chi2; p.status = out->status;
  p.nn = c->nn_on ? c->d_nn : nullptr; p.snx = seeds->nx; p.snuv = seeds->nuv; p.ghost = out->ghost;
  p.shits = seeds->hits;
  p.long_cap_total = (size_t)velo->n_events * (size_t)c->geom.max_long_per_event;
  if (c->match_threads == 128)
    lhcb::matching_kernel<128, 6><<<velo->n_events, 128, c->match_smem, (cudaStream_t)stream>>>(p);
  else
    lhcb::matching_kernel<256, 3><<<velo->n_events, 256, c->match_smem, (cudaStream_t)stream>>>(p);
  LHCB_CUDA(c, cudaGetLastError());
  c->last_launches = 1;
  return LHCB_OK;
}

const char* lhcb_error_string(int s) {
  switch (s) {
    case LHCB_OK: return "ok";
    case LHCB_ERR_BAD_ARGUMENT: return "bad argument";
    case LHCB_ERR_BAD_GEOMETRY: return "bad geometry";
    case LHCB_ERR_CUDA: return "CUDA runtime error";
    case LHCB_ERR_NOT_INITIALISED: return "context not initialised";
    case LHCB_ERR_CAPACITY: return "capacities exceed the shared memory of the device";
    default: return "unknown status";
  }
}

#ifdef LHCB_STAGE_CLOCKS
// diagnostic builds only: out[0..15] cycles summed over CTAs per stage, out[16..23] maxima over CTAs of the
// queue fills (lhcb::g_dbg_max); reset != 0 zeroes both
int lhcb_debug_stage_clocks(unsigned long long* out, int reset) {
  if (out) {
    if (cudaMemcpyFromSymbol(out, lhcb::g_stage_clk, sizeof(lhcb::g_stage_clk)) != cudaSuccess) return LHCB_ERR_CUDA;
    unsigned int m[8];
    if (cudaMemcpyFromSymbol(m, lhcb::g_dbg_max, sizeof(m)) != cudaSuccess) return LHCB_ERR_CUDA;
    for (int i = 0; i < 8; ++i) out[16 + i] = m[i];
  }
  if (reset) {
    unsigned long long z[16] = {0};
    unsigned int zm[8] = {0};
    if (cudaMemcpyToSymbol(lhcb::g_stage_clk, z, sizeof(z)) != cudaSuccess) return LHCB_ERR_CUDA;
    if (cudaMemcpyToSymbol(lhcb::g_dbg_max, zm, sizeof(zm)) != cudaSuccess) return LHCB_ERR_CUDA;
  }
  return LHCB_OK;
}
#endif

int lhcb_last_cuda_error(const lhcb_ctx* c) { return c ? c->last_cuda_error : 0; }
int lhcb_last_launch_count(const lhcb_ctx* c) { return c ? c->last_launches : 0; }
int lhcb_launch_config(const lhcb_ctx* c, int out[4]) {
  if (!c || !out) return LHCB_ERR_BAD_ARGUMENT;
  out[0] = c->seed_threads; out[1] = (int)c->seed_smem; out[2] = c->match_threads; out[3] = (int)c->match_smem;
  return LHCB_OK;
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// Host-buffer pipeline: slices of events, two streams, copies of one slice overlap kernels of another.
struct lhcb_pipeline {
  lhcb_ctx* ctx;
  int max_events, slice;
  size_t max_hits, max_velo, max_ut;
  cudaStream_t st[2];
  // inputs (whole batch, same offsets as on the host)
  uint32_t *zone_off, *velo_off, *ut_off;
  float *hit_x, *vx, *vy, *vtx, *vty, *ux, *uylo, *uyhi;
  int8_t* pol;
  // per-stream seeds and long-track buffers (one slice each)
  struct Slot {
    uint32_t *s_count, *s_hits, *s_status; float *s_state, *s_par; uint8_t *s_nx, *s_nuv;
    uint32_t *l_count, *l_seed, *l_velo, *l_ut, *l_status; uint8_t* l_nut; float *l_qop, *l_chi2;
  } slot[2];
  uint64_t h2d, d2h;
  int launches;
};

namespace {
template <class T>
cudaError_t dalloc(T** p, size_t n) { return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T)); }
}  // namespace

extern "C" {

void lhcb_pipeline_destroy(lhcb_pipeline* p) {
  if (!p) return;
  cudaSetDevice(p->ctx->device);
  for (int i = 0; i < 2; ++i) {
    if (p->st[i]) { cudaStreamSynchronize(p->st[i]); cudaStreamDestroy(p->st[i]); }
    lhcb_pipeline::Slot& s = p->slot[i];
    cudaFree(s.s_count); cudaFree(s.s_hits); cudaFree(s.s_status); cudaFree(s.s_state); cudaFree(s.s_par);
    cudaFree(s.s_nx); cudaFree(s.s_nuv); cudaFree(s.l_count); cudaFree(s.l_seed); cudaFree(s.l_velo);
    cudaFree(s.l_ut); cudaFree(s.l_status); cudaFree(s.l_nut); cudaFree(s.l_qop); cudaFree(s.l_chi2);
  }
  cudaFree(p->zone_off); cudaFree(p->velo_off); cudaFree(p->ut_off); cudaFree(p->hit_x); cudaFree(p->vx);
  cudaFree(p->vy); cudaFree(p->vtx); cudaFree(p->vty); cudaFree(p->ux); cudaFree(p->uylo); cudaFree(p->uyhi);
  cudaFree(p->pol);
  delete p;
}

int lhcb_pipeline_create(lhcb_ctx* c, int max_events, size_t max_hits, size_t max_velo, size_t max_ut,
                         int slice_events, lhcb_pipeline** out) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!out || max_events <= 0 || slice_events <= 0) return LHCB_ERR_BAD_ARGUMENT;
  *out = nullptr;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  lhcb_pipeline* p = new (std::nothrow) lhcb_pipeline();
  if (!p) return LHCB_ERR_BAD_ARGUMENT;
  std::memset(p, 0, sizeof(*p));
  p->ctx = c; p->max_events = max_events; p->slice = slice_events < max_events ? slice_events : max_events;
  p->max_hits = max_hits; p->max_velo = max_velo; p->max_ut = max_ut;
  const size_t ms = c->geom.max_seeds_per_half, ml = c->geom.max_long_per_event, sl = p->slice;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  for (int i = 0; i < 2; ++i) ok(cudaStreamCreateWithFlags(&p->st[i], cudaStreamNonBlocking));
  ok(dalloc(&p->zone_off, (size_t)max_events * 24 + 1)); ok(dalloc(&p->velo_off, (size_t)max_events + 1));
  ok(dalloc(&p->ut_off, (size_t)max_events * 4 + 1)); ok(dalloc(&p->hit_x, max_hits + 4));
  ok(dalloc(&p->vx, max_velo)); ok(dalloc(&p->vy, max_velo)); ok(dalloc(&p->vtx, max_velo)); ok(dalloc(&p->vty, max_velo));
  ok(dalloc(&p->ux, max_ut)); ok(dalloc(&p->uylo, max_ut)); ok(dalloc(&p->uyhi, max_ut));
  ok(dalloc(&p->pol, (size_t)max_events));
  for (int i = 0; i < 2; ++i) {
    lhcb_pipeline::Slot& s = p->slot[i];
    const size_t cs = sl * 2 * ms, cl = sl * ml;
    ok(dalloc(&s.s_count, sl * 2)); ok(dalloc(&s.s_status, sl * 2)); ok(dalloc(&s.s_state, 5 * cs));
    ok(dalloc(&s.s_par, 7 * cs)); ok(dalloc(&s.s_hits, 12 * cs)); ok(dalloc(&s.s_nx, cs)); ok(dalloc(&s.s_nuv, cs));
    ok(dalloc(&s.l_count, sl)); ok(dalloc(&s.l_status, sl)); ok(dalloc(&s.l_seed, cl)); ok(dalloc(&s.l_velo, cl));
    ok(dalloc(&s.l_ut, 4 * cl)); ok(dalloc(&s.l_nut, cl)); ok(dalloc(&s.l_qop, cl)); ok(dalloc(&s.l_chi2, cl));
  }
  if (e != cudaSuccess) { c->last_cuda_error = (int)e; lhcb_pipeline_destroy(p); return LHCB_ERR_CUDA; }
  *out = p;
  return LHCB_OK;
}

int lhcb_reconstruct_host(lhcb_pipeline* p, const lhcb_events_t* ev, const lhcb_velo_t* velo, const lhcb_ut_t* ut,
                          lhcb_long_t* out, uint32_t* host_seed_count) {
  if (!p) return LHCB_ERR_NOT_INITIALISED;
  lhcb_ctx* c = p->ctx;
  if (!ev || !velo || !out || ev->n_events < 0 || velo->n_events != ev->n_events || !ev->zone_off || !velo->off ||
      !out->count || !out->seed_idx || !out->velo_idx || !out->ut_idx || !out->n_ut || !out->qop || !out->chi2 ||
      !out->status)
    return LHCB_ERR_BAD_ARGUMENT;
  const int n = ev->n_events;
  p->h2d = p->d2h = 0; p->launches = 0;
  if (n == 0) return LHCB_OK;
  if (n > p->max_events || ev->n_hits > p->max_hits) return LHCB_ERR_CAPACITY;
  const size_t n_velo = velo->off[n];
  const size_t n_ut = ut ? ut->off[(size_t)n * 4] : 0;
  if (n_velo > p->max_velo || n_ut > p->max_ut) return LHCB_ERR_CAPACITY;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  const size_t ms = c->geom.max_seeds_per_half, ml = c->geom.max_long_per_event;
  const size_t ct_all = (size_t)n * ml;
  auto H2D = [&](void* d, const void* h, size_t bytes, cudaStream_t s) {
    p->h2d += bytes;
    return bytes ? cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, s) : cudaSuccess;
  };
  auto D2H = [&](void* h, const void* d, size_t bytes, cudaStream_t s) {
    p->d2h += bytes;
    return bytes ? cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, s) : cudaSuccess;
  };
  int k = 0;
  for (int e0 = 0; e0 < n; e0 += p->slice, ++k) {
    const int ne = (n - e0) < p->slice ? (n - e0) : p->slice;
    cudaStream_t s = p->st[k & 1];
    lhcb_pipeline::Slot& S = p->slot[k & 1];
    // ---- inputs of this slice, at the same offsets as on the host
    const size_t z0 = (size_t)e0 * 24, z1 = (size_t)(e0 + ne) * 24;
    const size_t h0 = ev->zone_off[z0], h1 = ev->zone_off[z1];
    const size_t v0 = velo->off[e0], v1 = velo->off[e0 + ne];
    LHCB_CUDA(c, H2D(p->zone_off + z0, ev->zone_off + z0, (z1 - z0 + 1) * 4, s));
    LHCB_CUDA(c, H2D(p->hit_x + h0, ev->hit_x + h0, (h1 - h0) * 4, s));
    if (ev->polarity) LHCB_CUDA(c, H2D(p->pol + e0, ev->polarity + e0, (size_t)ne, s));
    LHCB_CUDA(c, H2D(p->velo_off + e0, velo->off + e0, ((size_t)ne + 1) * 4, s));
    LHCB_CUDA(c, H2D(p->vx + v0, velo->x + v0, (v1 - v0) * 4, s));
    LHCB_CUDA(c, H2D(p->vy + v0, velo->y + v0, (v1 - v0) * 4, s));
    LHCB_CUDA(c, H2D(p->vtx + v0, velo->tx + v0, (v1 - v0) * 4, s));
    LHCB_CUDA(c, H2D(p->vty + v0, velo->ty + v0, (v1 - v0) * 4, s));
    if (ut) {
      const size_t u0 = ut->off[(size_t)e0 * 4], u1 = ut->off[(size_t)(e0 + ne) * 4];
      LHCB_CUDA(c, H2D(p->ut_off + (size_t)e0 * 4, ut->off + (size_t)e0 * 4, ((size_t)ne * 4 + 1) * 4, s));
      LHCB_CUDA(c, H2D(p->ux + u0, ut->x0 + u0, (u1 - u0) * 4, s));
      LHCB_CUDA(c, H2D(p->uylo + u0, ut->y_lo + u0, (u1 - u0) * 4, s));
      LHCB_CUDA(c, H2D(p->uyhi + u0, ut->y_hi + u0, (u1 - u0) * 4, s));
    }
    // ---- kernels
    lhcb_events_t dev_ev = {ne, (uint32_t)p->max_hits, p->zone_off + z0, p->hit_x, ev->polarity ? p->pol + e0 : nullptr};
    dev_ev.n_hits = ev->n_hits;
    lhcb_seeds_t dev_s = {ne, S.s_count, S.s_state, S.s_par, S.s_hits, S.s_nx, S.s_nuv, S.s_status};
    int rc = lhcb_seeding(c, &dev_ev, &dev_s, nullptr, s);
    if (rc != LHCB_OK) return rc;
    p->launches += c->last_launches;
    lhcb_velo_t dev_v = {ne, p->velo_off + e0, p->vx, p->vy, p->vtx, p->vty, ev->polarity ? p->pol + e0 : nullptr};
    lhcb_ut_t dev_u = {(uint32_t)n_ut, p->ut_off + (size_t)e0 * 4, p->ux, p->uylo, p->uyhi};
    lhcb_long_t dev_l = {S.l_count, S.l_seed, S.l_velo, S.l_ut, S.l_nut, S.l_qop, S.l_chi2, S.l_status, nullptr};
    rc = lhcb_matching(c, &dev_s, &dev_v, ut ? &dev_u : nullptr, &dev_l, nullptr, s);
    if (rc != LHCB_OK) return rc;
    p->launches += c->last_launches;
    // ---- outputs of this slice
    const size_t o = (size_t)e0 * ml, cl = (size_t)ne * ml;
    LHCB_CUDA(c, D2H(out->count + e0, S.l_count, (size_t)ne * 4, s));
    LHCB_CUDA(c, D2H(out->status + e0, S.l_status, (size_t)ne * 4, s));
    LHCB_CUDA(c, D2H(out->seed_idx + o, S.l_seed, cl * 4, s));
    LHCB_CUDA(c, D2H(out->velo_idx + o, S.l_velo, cl * 4, s));
    for (int l = 0; l < 4; ++l) LHCB_CUDA(c, D2H(out->ut_idx + (size_t)l * ct_all + o, S.l_ut + (size_t)l * cl, cl * 4, s));
    LHCB_CUDA(c, D2H(out->n_ut + o, S.l_nut, cl, s));
    LHCB_CUDA(c, D2H(out->qop + o, S.l_qop, cl * 4, s));
    LHCB_CUDA(c, D2H(out->chi2 + o, S.l_chi2, cl * 4, s));
    if (host_seed_count) LHCB_CUDA(c, D2H(host_seed_count + (size_t)e0 * 2, S.s_count, (size_t)ne * 8, s));
  }
  LHCB_CUDA(c, cudaStreamSynchronize(p->st[0]));
  LHCB_CUDA(c, cudaStreamSynchronize(p->st[1]));
  (void)ms;
  return LHCB_OK;
}

int lhcb_pipeline_last_bytes(const lhcb_pipeline* p, uint64_t* h2d, uint64_t* d2h) {
  if (!p) return LHCB_ERR_NOT_INITIALISED;
  if (h2d) *h2d = p->h2d;
  if (d2h) *d2h = p->d2h;
  return p->launches;
}

}  // extern "C"
