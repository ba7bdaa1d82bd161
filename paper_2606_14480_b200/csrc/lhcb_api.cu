// C-ABI entry points (include/lhcb.h): argument checks, constant derivation, kernel launches.
// No torch types: plain pointers and sizes.  Built with
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false -shared -Xcompiler -fPIC
#include <cuda_runtime.h>

#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include "../../include/lhcb.h"
#include "derive.h"
#include "matching.cuh"
#include "prepare.cuh"
#include "schedule.cuh"
#include "seeding.cuh"


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
  int prep_variant;   // instantiation of prepare_kernel (threads x hits per thread) that covers the event capacity
  int match_threads;  // 128 when six CTAs fit an SM, else 256
  int seed_threads;   // 256 when four CTAs fit the SM's shared memory, else 512
  int seed_ctas;      // CTAs per SM the seeding kernel is compiled for (register budget)
  int last_cuda_error;
  int last_launches;
  // the last launch made through this context, when it was a Seeding with lhcb_order's workspace: only the
  // lhcb_matching call that follows it directly, on the same stream, workspace and batch size, may be launched as
  // its programmatic dependent (the per-half flags the Matching waits on are lowered and raised by THAT grid)
  const void* pdl_ws;
  const void* pdl_stream;
  int pdl_events;
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
      G.max_velo_per_event > 65535 || G.max_ut_per_event > 65534 || G.max_match_cand_per_event > 16383 || G.max_triplets_per_half < G.max_xz_cand_per_half) { delete c; return LHCB_ERR_BAD_ARGUMENT; }
  // 256-thread CTAs, four per SM, when their shared memory fits (228 KB per SM, 1 KB reserved per
  // CTA); else 512-thread CTAs, two (or one) per SM
  c->seed_threads = 256;
  c->seed_smem = lhcb::seed_smem_bytes(G.max_hits_per_half, G.max_xz_cand_per_half, G.max_triplets_per_half);
  // 256-thread CTAs, five per SM (48 registers per thread) or four (64), when their shared memory fits (228 KB
  // per SM, 1 KB reserved per CTA); else 512-thread CTAs, two (or one) per SM.  Five CTAs measured 7% faster
  // than four on the nominal workload: the kernel is bound by latency, more resident warps hide more of it.
  c->seed_ctas = 5;
  if (c->seed_smem > (size_t)(228 * 1024 / 5 - 1024)) c->seed_ctas = 4;
  if (c->seed_smem > (size_t)(228 * 1024 / 4 - 1024)) { c->seed_threads = 512; c->seed_ctas = 2; }
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
    const void* fn = c->seed_ctas == 5 ? (const void*)lhcb::seeding_kernel<256, 5>
                   : c->seed_ctas == 4 ? (const void*)lhcb::seeding_kernel<256, 4>
                                       : (const void*)lhcb::seeding_kernel<512, 2>;
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->seed_smem);
  }
  if (e == cudaSuccess)
    e = c->match_threads == 128
            ? cudaFuncSetAttribute(lhcb::matching_kernel<128, 6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->match_smem)
            : cudaFuncSetAttribute(lhcb::matching_kernel<256, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->match_smem);
  // the preparation keeps one register per raw hit: T threads x R hits per thread >= the event capacity
  c->prep_variant = 2 * G.max_hits_per_half <= 512 * 12 ? 0 : 2 * G.max_hits_per_half <= 1024 * 12 ? 1 : 2;
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(c->prep_variant == 0   ? (const void*)lhcb::prepare_kernel<512, 12, 4>
                             : c->prep_variant == 1 ? (const void*)lhcb::prepare_kernel<1024, 12, 1>
                                                    : (const void*)lhcb::prepare_kernel<1024, 16, 1>,
                             cudaFuncAttributeMaxDynamicSharedMemorySize, (int)c->prep_smem);
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
  (void)c; (void)n_scifi_hits;
  // every intermediate of the two kernels lives in shared memory; the workspace holds only the optional CTA
  // orders of lhcb_order: u32[2 n_events] for the Seeding, u32[n_events] for the Matching
  // and u32[2 n_events] "seeds are in global memory" flags
  return n_events > 0 ? (((size_t)n_events * 20 + 15) & ~(size_t)15) : 0;
}

int lhcb_order(lhcb_ctx* c, const lhcb_events_t* ev, const lhcb_velo_t* velo, const lhcb_ut_t* ut, void* workspace,
               void* stream) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!ev || !workspace || ev->n_events < 0 || (velo && velo->n_events != ev->n_events)) return LHCB_ERR_BAD_ARGUMENT;
  c->last_launches = 0;
  c->pdl_ws = nullptr;
  if (ev->n_events == 0) return LHCB_OK;
  if (!ev->zone_off || (velo && !velo->off) || (ut && !ut->off)) return LHCB_ERR_BAD_ARGUMENT;
  // a large batch is dozens of waves of CTAs: its tail is a small part of the run, and both the sorted order and
  // the per-half flags measured about 1% slower than the plain launches (16,384 events): nothing to do, and
  // lhcb_seeding / lhcb_matching ignore the workspace for such a batch
  if (ev->n_events > lhcb::kOrderMaxSorted) return LHCB_OK;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  uint32_t* so = static_cast<uint32_t*>(workspace);
  lhcb::order_kernel<<<1, lhcb::kOrderThreads, 0, (cudaStream_t)stream>>>(ev->n_events, ev->zone_off, ut ? ut->off : nullptr,
                                                                        velo ? velo->off : nullptr, so,
                                                                        so + (size_t)ev->n_events * 2,   // identity without velo and ut
                                                                        so + (size_t)ev->n_events * 3);
  LHCB_CUDA(c, cudaGetLastError());
  c->last_launches = 1;
  return LHCB_OK;
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
  c->pdl_ws = nullptr;
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
  if (c->prep_variant == 0) lhcb::prepare_kernel<512, 12, 4><<<raw->n_events, 512, c->prep_smem, (cudaStream_t)stream>>>(p);
  else if (c->prep_variant == 1) lhcb::prepare_kernel<1024, 12, 1><<<raw->n_events, 1024, c->prep_smem, (cudaStream_t)stream>>>(p);
  else lhcb::prepare_kernel<1024, 16, 1><<<raw->n_events, 1024, c->prep_smem, (cudaStream_t)stream>>>(p);
  LHCB_CUDA(c, cudaGetLastError());
  c->last_launches = 1;
  return LHCB_OK;
}

int lhcb_seeding(lhcb_ctx* c, const lhcb_events_t* ev, lhcb_seeds_t* out, void* workspace, void* stream) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!ev || !out || ev->n_events < 0) return LHCB_ERR_BAD_ARGUMENT;
  c->last_launches = 0;
  c->pdl_ws = nullptr;
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
  if (ev->n_events > lhcb::kOrderMaxSorted) workspace = nullptr;
  p.order = static_cast<const uint32_t*>(workspace);        // CTA order of lhcb_order, or NULL: CTA b takes half b
  p.done = workspace ? static_cast<uint32_t*>(workspace) + (size_t)ev->n_events * 3 : nullptr;
  if (c->seed_ctas == 5)
    lhcb::seeding_kernel<256, 5><<<ev->n_events * 2, 256, c->seed_smem, (cudaStream_t)stream>>>(p);
  else if (c->seed_ctas == 4)
    lhcb::seeding_kernel<256, 4><<<ev->n_events * 2, 256, c->seed_smem, (cudaStream_t)stream>>>(p);
  else
    lhcb::seeding_kernel<512, 2><<<ev->n_events * 2, 512, c->seed_smem, (cudaStream_t)stream>>>(p);
  LHCB_CUDA(c, cudaGetLastError());
  c->last_launches = 1;
  if (workspace) { c->pdl_ws = workspace; c->pdl_stream = stream; c->pdl_events = ev->n_events; }
  return LHCB_OK;
}

int lhcb_matching(lhcb_ctx* c, const lhcb_seeds_t* seeds, const lhcb_velo_t* velo, const lhcb_ut_t* ut,
                  lhcb_long_t* out, void* workspace, void* stream) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!seeds || !velo || !out || velo->n_events < 0 || seeds->n_events != velo->n_events)
    return LHCB_ERR_BAD_ARGUMENT;
  c->last_launches = 0;
  // programmatic dependent launch only straight after the Seeding launch whose flags this grid will wait on
  const bool after_seeding = workspace && c->pdl_ws == workspace && c->pdl_stream == stream && c->pdl_events == velo->n_events;
  c->pdl_ws = nullptr;
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
  if (velo->n_events > lhcb::kOrderMaxSorted) workspace = nullptr;
  p.order = workspace ? static_cast<const uint32_t*>(workspace) + (size_t)velo->n_events * 2 : nullptr;
  p.done = workspace ? static_cast<const uint32_t*>(workspace) + (size_t)velo->n_events * 3 : nullptr;
  p.long_cap_total = (size_t)velo->n_events * (size_t)c->geom.max_long_per_event;
  {
    // straight after a Seeding launch with the same workspace, the launch is a programmatic dependent of that grid:
    // its CTAs may start while the last Seeding wave drains and wait for their event's flags.  After anything else
    // (lhcb_order alone, given seeds, another call in between) it is an ordinary launch: the kernel has no
    // griddepcontrol.wait, so nothing but those flags would order it against a still-running predecessor
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((unsigned)velo->n_events); cfg.blockDim = dim3((unsigned)c->match_threads);
    cfg.dynamicSmemBytes = c->match_smem; cfg.stream = (cudaStream_t)stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = (workspace && after_seeding) ? 1 : 0;
    if (c->match_threads == 128) LHCB_CUDA(c, cudaLaunchKernelEx(&cfg, lhcb::matching_kernel<128, 6>, p));
    else LHCB_CUDA(c, cudaLaunchKernelEx(&cfg, lhcb::matching_kernel<256, 3>, p));
  }
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
    case LHCB_ERR_STATIC_SCRATCH:
      return "batch has more events than the built-in scratch of lhcb_seeding_static holds (LHCB_STATIC_MAX_EVENTS = 3072): "
             "split the batch, or use lhcb_order + lhcb_seeding with a workspace of your own";
    default: return "unknown status";
  }
}

#ifdef LHCB_CHECKED
namespace lhcb {
__global__ void check_selftest_kernel(int i, int n) { LHCB_CHECK_IDX(i, n); }
}  // namespace lhcb
// one deliberate check of index i against bound n on the device: the test of the checker itself
int lhcb_debug_check_selftest(int i, int n) {
  lhcb::check_selftest_kernel<<<1, 1>>>(i, n);
  return cudaDeviceSynchronize() == cudaSuccess ? LHCB_OK : LHCB_ERR_CUDA;
}
// diagnostic build only (-DLHCB_CHECKED): out = {failed index checks, source line of the first failure, its index,
// its bound, checks made (low word), checks made (high word)}; reset != 0 zeroes the counters
int lhcb_debug_checks(unsigned int* out, int reset) {
  if (out) {
    unsigned long long n = 0;
    if (cudaMemcpyFromSymbol(out, lhcb::g_check, sizeof(lhcb::g_check)) != cudaSuccess) return LHCB_ERR_CUDA;
    if (cudaMemcpyFromSymbol(&n, lhcb::g_check_count, sizeof(n)) != cudaSuccess) return LHCB_ERR_CUDA;
    out[4] = (unsigned int)n; out[5] = (unsigned int)(n >> 32);
  }
  if (reset) {
    const unsigned int z[4] = {0, 0, 0, 0};
    const unsigned long long zn = 0;
    if (cudaMemcpyToSymbol(lhcb::g_check, z, sizeof(z)) != cudaSuccess) return LHCB_ERR_CUDA;
    if (cudaMemcpyToSymbol(lhcb::g_check_count, &zn, sizeof(zn)) != cudaSuccess) return LHCB_ERR_CUDA;
  }
  return LHCB_OK;
}
#endif
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
// lhcb_seeding_static (include/lhcb.h): the heaviest-first Seeding for callers that cannot bring a workspace.
// The CTA order and the per-half flags that lhcb_order / lhcb_seeding keep in a caller-owned workspace live
// here in an array that is part of the library image: the driver places it when the module is loaded on a
// device and it stays there until the process exits, so no call ever allocates or frees for it.
namespace {
// same layout as lhcb_workspace_bytes: 5 words per event (Seeding order [2n], Matching order [n], flags [2n])
static __device__ __align__(256) uint32_t g_static_ws[(size_t)LHCB_STATIC_MAX_EVENTS * 5];   // 61,440 bytes per device
static_assert(LHCB_STATIC_MAX_EVENTS <= lhcb::kOrderMaxSorted, "lhcb_seeding ignores a workspace above kOrderMaxSorted events");

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_addr[kStaticMaxDevices];   // device address of g_static_ws on each device, once looked up

// `g_static_ws` in host code names a host-side handle, not the memory the kernels see: its device address has to
// be asked for, with the device current, once per device (each device holds its own copy of the array).
cudaError_t static_ws_address(int device, void** out) {
  std::lock_guard<std::mutex> lock(g_static_mu);
  if (device < kStaticMaxDevices && g_static_addr[device]) { *out = g_static_addr[device]; return cudaSuccess; }
  void* a = nullptr;
  const cudaError_t e = cudaGetSymbolAddress(&a, g_static_ws);
  if (e != cudaSuccess) return e;
  if (!a) return cudaErrorInvalidSymbol;
  if (device < kStaticMaxDevices) g_static_addr[device] = a;
  *out = a;
  return cudaSuccess;
}
}  // namespace

extern "C" int lhcb_seeding_static(lhcb_ctx* c, const lhcb_events_t* ev, lhcb_seeds_t* out, void* stream) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!ev || !out || ev->n_events < 0) return LHCB_ERR_BAD_ARGUMENT;
  if (ev->n_events > LHCB_STATIC_MAX_EVENTS) return LHCB_ERR_STATIC_SCRATCH;   // nothing is launched
  c->last_launches = 0;
  if (ev->n_events == 0) return LHCB_OK;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  void* ws = nullptr;
  LHCB_CUDA(c, static_ws_address(c->device, &ws));
  // order_kernel rewrites every word of the array that belongs to this batch (orders [0, 3n), flags [3n, 5n)),
  // so what the previous call left behind is never seen; nothing has to start at zero
  int rc = lhcb_order(c, ev, nullptr, nullptr, ws, stream);
  if (rc != LHCB_OK) return rc;
  rc = lhcb_seeding(c, ev, out, ws, stream);
  c->pdl_ws = nullptr;                                       // the array is private: no Matching is ever its dependent
  if (rc != LHCB_OK) return rc;
  c->last_launches = 2;
  return LHCB_OK;
}

// ---------------------------------------------------------------------------------------------
// Host-buffer pipeline: slices of events on three streams (H2D copies, kernels, D2H copies).  The kernels of
// a slice (order, seeding, matching, compaction) are captured once in a CUDA graph and replayed.
struct lhcb_pipeline {
  lhcb_ctx* ctx;
  int max_events, slice, n_slices;
  size_t max_hits, max_velo, max_ut;
  uint32_t cap_s, cap_l;
  cudaStream_t st_in, st_k, st_out;
  cudaEvent_t *ev_in, *ev_k;          // per slice
  // inputs (whole batch, same offsets as on the host)
  uint32_t *zone_off, *velo_off, *ut_off;
  float *hit_x, *vx, *vy, *vtx, *vty, *ux;
  uint8_t* urow;
  uint16_t* ustrip;
  int8_t* pol;
  // slot buffers of one slice (lhcb_seeds_t / lhcb_long_t layout)
  uint32_t *s_count, *s_hits, *s_status; float *s_state, *s_par; uint8_t *s_nx, *s_nuv;
  uint32_t *l_count, *l_seed, *l_velo, *l_ut, *l_status; uint8_t* l_nut; float *l_qop, *l_chi2;
  void* order_ws;
  // dense outputs of the whole batch
  uint32_t *d_s_off, *d_l_off, *d_s_status, *d_l_status;
  float *d_state, *d_par; uint16_t* d_hits; uint8_t *d_nx, *d_nuv;
  uint32_t *d_seed, *d_velo, *d_ut; uint8_t* d_nut; float *d_qop, *d_chi2;
  uint32_t *totals, *slice_totals;    // device: [2], [n_slices][4]
  uint32_t* h_totals;                 // pinned host mirror of slice_totals
  // one graph per slice
  struct Graph { cudaGraphExec_t exec; int e0, ne; unsigned flags; int launches; } * graphs;
  int* e0;                            // [n_slices + 1] first event of each slice of the current batch
  uint64_t h2d, d2h;
  int launches;
};

namespace {
template <class T>
cudaError_t dalloc(T** p, size_t n) { return cudaMalloc((void**)p, (n ? n : 1) * sizeof(T)); }

// the kernels of one slice on the compute stream (captured into the slice's graph)
int enqueue_slice(lhcb_pipeline* p, int k, int e0, int ne, bool has_ut, bool has_pol, bool want_par, bool strips,
                  int* launches) {
  lhcb_ctx* c = p->ctx;
  cudaStream_t s = p->st_k;
  *launches = (has_ut && strips) ? 1 : 0;
  if (has_ut && strips)                                      // the slice's UT hits arrived as strip numbers
    lhcb::ut_decode_kernel<<<296, 256, 0, s>>>(p->ut_off + (size_t)e0 * 4, p->ut_off + (size_t)(e0 + ne) * 4, p->ustrip, p->ux,
                                               c->geom.ut_strip_x0, c->geom.ut_strip_pitch);
  const size_t z0 = (size_t)e0 * 24;
  lhcb_events_t dev_ev = {ne, (uint32_t)p->max_hits, p->zone_off + z0, p->hit_x, has_pol ? p->pol + e0 : nullptr};
  lhcb_velo_t dev_v = {ne, p->velo_off + e0, p->vx, p->vy, p->vtx, p->vty, has_pol ? p->pol + e0 : nullptr};
  lhcb_ut_t dev_u = {(uint32_t)p->max_ut, p->ut_off + (size_t)e0 * 4, p->ux, nullptr, nullptr, p->urow};
  lhcb_seeds_t dev_s = {ne, p->s_count, p->s_state, p->s_par, p->s_hits, p->s_nx, p->s_nuv, p->s_status};
  lhcb_long_t dev_l = {p->l_count, p->l_seed, p->l_velo, p->l_ut, p->l_nut, p->l_qop, p->l_chi2, p->l_status, nullptr};
  int rc = lhcb_order(c, &dev_ev, &dev_v, has_ut ? &dev_u : nullptr, p->order_ws, s);
  if (rc != LHCB_OK) return rc;
  *launches += c->last_launches;                             // 0 for a slice above kOrderMaxSorted events
  rc = lhcb_seeding(c, &dev_ev, &dev_s, p->order_ws, s);
  if (rc != LHCB_OK) return rc;
  *launches += c->last_launches;
  rc = lhcb_matching(c, &dev_s, &dev_v, has_ut ? &dev_u : nullptr, &dev_l, p->order_ws, s);
  if (rc != LHCB_OK) return rc;
  *launches += c->last_launches + 2;                         // + the two compaction kernels below
  lhcb::CompactParams q;
  std::memset(&q, 0, sizeof(q));
  q.n_events = ne; q.max_seeds = c->geom.max_seeds_per_half; q.max_long = c->geom.max_long_per_event;
  q.s_count = p->s_count; q.s_state = p->s_state; q.s_par = p->s_par; q.s_hits = p->s_hits; q.s_nx = p->s_nx; q.s_nuv = p->s_nuv;
  q.l_count = p->l_count; q.l_seed = p->l_seed; q.l_velo = p->l_velo; q.l_ut = p->l_ut; q.l_nut = p->l_nut;
  q.l_qop = p->l_qop; q.l_chi2 = p->l_chi2;
  q.totals = p->totals; q.slice_totals = p->slice_totals + (size_t)k * 4;
  q.s_off = p->d_s_off + (size_t)e0 * 2; q.l_off = p->d_l_off + e0;
  q.cap_s = p->cap_s; q.cap_l = p->cap_l;
  q.d_state = p->d_state; q.d_par = want_par ? p->d_par : nullptr; q.d_hits = p->d_hits; q.zone_off = p->zone_off + z0; q.d_nx = p->d_nx; q.d_nuv = p->d_nuv;
  q.d_seed = p->d_seed; q.d_velo = p->d_velo; q.d_ut = p->d_ut; q.d_nut = p->d_nut; q.d_qop = p->d_qop; q.d_chi2 = p->d_chi2;
  lhcb::compact_scan_kernel<<<2, lhcb::kScanThreads, 0, s>>>(q);
  const int groups = 3 * ne, per = lhcb::kGatherThreads / 32;
  lhcb::compact_gather_kernel<<<(groups + per - 1) / per, lhcb::kGatherThreads, 0, s>>>(q);
  LHCB_CUDA(c, cudaGetLastError());
  // status words of the slice into the batch arrays, totals to the host mirror
  LHCB_CUDA(c, cudaMemcpyAsync(p->d_s_status + (size_t)e0 * 2, p->s_status, (size_t)ne * 8, cudaMemcpyDeviceToDevice, s));
  LHCB_CUDA(c, cudaMemcpyAsync(p->d_l_status + e0, p->l_status, (size_t)ne * 4, cudaMemcpyDeviceToDevice, s));
  LHCB_CUDA(c, cudaMemcpyAsync(p->h_totals + (size_t)k * 4, p->slice_totals + (size_t)k * 4, 16, cudaMemcpyDeviceToHost, s));
  return LHCB_OK;
}
}  // namespace

extern "C" {

void lhcb_pipeline_destroy(lhcb_pipeline* p) {
  if (!p) return;
  cudaSetDevice(p->ctx->device);
  for (cudaStream_t s : {p->st_in, p->st_k, p->st_out})
    if (s) { cudaStreamSynchronize(s); cudaStreamDestroy(s); }
  for (int k = 0; k < p->n_slices; ++k) {
    if (p->ev_in && p->ev_in[k]) cudaEventDestroy(p->ev_in[k]);
    if (p->ev_k && p->ev_k[k]) cudaEventDestroy(p->ev_k[k]);
    if (p->graphs && p->graphs[k].exec) cudaGraphExecDestroy(p->graphs[k].exec);
  }
  delete[] p->ev_in; delete[] p->ev_k; delete[] p->graphs; delete[] p->e0;
  for (void* q : {(void*)p->zone_off, (void*)p->velo_off, (void*)p->ut_off, (void*)p->hit_x, (void*)p->vx, (void*)p->vy,
                  (void*)p->vtx, (void*)p->vty, (void*)p->ux, (void*)p->urow, (void*)p->ustrip, (void*)p->pol, (void*)p->s_count,
                  (void*)p->s_hits, (void*)p->s_status, (void*)p->s_state, (void*)p->s_par, (void*)p->s_nx, (void*)p->s_nuv,
                  (void*)p->l_count, (void*)p->l_seed, (void*)p->l_velo, (void*)p->l_ut, (void*)p->l_status, (void*)p->l_nut,
                  (void*)p->l_qop, (void*)p->l_chi2, p->order_ws, (void*)p->d_s_off, (void*)p->d_l_off, (void*)p->d_s_status,
                  (void*)p->d_l_status, (void*)p->d_state, (void*)p->d_par, (void*)p->d_hits, (void*)p->d_nx, (void*)p->d_nuv,
                  (void*)p->d_seed, (void*)p->d_velo, (void*)p->d_ut, (void*)p->d_nut, (void*)p->d_qop, (void*)p->d_chi2,
                  (void*)p->totals, (void*)p->slice_totals})
    cudaFree(q);
  if (p->h_totals) cudaFreeHost(p->h_totals);
  delete p;
}

int lhcb_pipeline_create(lhcb_ctx* c, int max_events, size_t max_hits, size_t max_velo, size_t max_ut,
                         int slice_events, size_t max_seeds_total, size_t max_long_total, lhcb_pipeline** out) {
  if (!c) return LHCB_ERR_NOT_INITIALISED;
  if (!out || max_events <= 0 || slice_events <= 0 || max_seeds_total > 0xFFFFFFF0u || max_long_total > 0xFFFFFFF0u)
    return LHCB_ERR_BAD_ARGUMENT;
  *out = nullptr;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  lhcb_pipeline* p = new (std::nothrow) lhcb_pipeline();
  if (!p) return LHCB_ERR_BAD_ARGUMENT;
  std::memset(p, 0, sizeof(*p));
  p->ctx = c; p->max_events = max_events; p->slice = slice_events < max_events ? slice_events : max_events;
  p->n_slices = (max_events + p->slice - 1) / p->slice + 3;   // the last slice is cut in up to four pieces (shorter tail)
  p->max_hits = max_hits; p->max_velo = max_velo; p->max_ut = max_ut;
  const size_t ms = c->geom.max_seeds_per_half, ml = c->geom.max_long_per_event, sl = p->slice;
  p->cap_s = (uint32_t)(max_seeds_total ? max_seeds_total : (size_t)max_events * 2 * ms);
  p->cap_l = (uint32_t)(max_long_total ? max_long_total : (size_t)max_events * ml);
  const size_t cs = sl * 2 * ms, cl = sl * ml, CS = p->cap_s, CL = p->cap_l;
  cudaError_t e = cudaSuccess;
  auto ok = [&](cudaError_t r) { if (e == cudaSuccess) e = r; };
  for (cudaStream_t* s : {&p->st_in, &p->st_k, &p->st_out}) ok(cudaStreamCreateWithFlags(s, cudaStreamNonBlocking));
  p->ev_in = new (std::nothrow) cudaEvent_t[p->n_slices]();
  p->ev_k = new (std::nothrow) cudaEvent_t[p->n_slices]();
  p->graphs = new (std::nothrow) lhcb_pipeline::Graph[p->n_slices]();
  p->e0 = new (std::nothrow) int[p->n_slices + 1]();
  if (!p->ev_in || !p->ev_k || !p->graphs || !p->e0) { lhcb_pipeline_destroy(p); return LHCB_ERR_BAD_ARGUMENT; }
  for (int k = 0; k < p->n_slices; ++k) {
    ok(cudaEventCreateWithFlags(&p->ev_in[k], cudaEventDisableTiming));
    ok(cudaEventCreateWithFlags(&p->ev_k[k], cudaEventDisableTiming));
  }
  ok(dalloc(&p->zone_off, (size_t)max_events * 24 + 1)); ok(dalloc(&p->velo_off, (size_t)max_events + 1));
  ok(dalloc(&p->ut_off, (size_t)max_events * 4 + 1)); ok(dalloc(&p->hit_x, max_hits + 8));
  ok(dalloc(&p->vx, max_velo)); ok(dalloc(&p->vy, max_velo)); ok(dalloc(&p->vtx, max_velo)); ok(dalloc(&p->vty, max_velo));
  ok(dalloc(&p->ux, max_ut + 8)); ok(dalloc(&p->urow, max_ut + 32)); ok(dalloc(&p->ustrip, max_ut + 8)); ok(dalloc(&p->pol, (size_t)max_events));
  ok(dalloc(&p->s_count, sl * 2)); ok(dalloc(&p->s_status, sl * 2)); ok(dalloc(&p->s_state, 5 * cs));
  ok(dalloc(&p->s_par, 7 * cs)); ok(dalloc(&p->s_hits, 12 * cs)); ok(dalloc(&p->s_nx, cs)); ok(dalloc(&p->s_nuv, cs));
  ok(dalloc(&p->l_count, sl)); ok(dalloc(&p->l_status, sl)); ok(dalloc(&p->l_seed, cl)); ok(dalloc(&p->l_velo, cl));
  ok(dalloc(&p->l_ut, 4 * cl)); ok(dalloc(&p->l_nut, cl)); ok(dalloc(&p->l_qop, cl)); ok(dalloc(&p->l_chi2, cl));
  ok(cudaMalloc(&p->order_ws, lhcb_workspace_bytes(c, (int)sl, 0) + 16));
  ok(dalloc(&p->d_s_off, (size_t)max_events * 2 + 1)); ok(dalloc(&p->d_l_off, (size_t)max_events + 1));
  ok(dalloc(&p->d_s_status, (size_t)max_events * 2)); ok(dalloc(&p->d_l_status, (size_t)max_events));
  ok(dalloc(&p->d_state, 5 * CS)); ok(dalloc(&p->d_par, 7 * CS)); ok(dalloc(&p->d_hits, 12 * CS));
  ok(dalloc(&p->d_nx, CS)); ok(dalloc(&p->d_nuv, CS));
  ok(dalloc(&p->d_seed, CL)); ok(dalloc(&p->d_velo, CL)); ok(dalloc(&p->d_ut, 4 * CL)); ok(dalloc(&p->d_nut, CL));
  ok(dalloc(&p->d_qop, CL)); ok(dalloc(&p->d_chi2, CL));
  ok(dalloc(&p->totals, 2)); ok(dalloc(&p->slice_totals, (size_t)p->n_slices * 4));
  ok(cudaMallocHost((void**)&p->h_totals, (size_t)p->n_slices * 16));
  if (e != cudaSuccess) { c->last_cuda_error = (int)e; lhcb_pipeline_destroy(p); return LHCB_ERR_CUDA; }
  *out = p;
  return LHCB_OK;
}

int lhcb_reconstruct_host(lhcb_pipeline* p, const lhcb_events_t* ev, const lhcb_velo_t* velo, const lhcb_ut_t* ut,
                          lhcb_host_seeds_t* so, lhcb_host_long_t* lo) {
  if (!p) return LHCB_ERR_NOT_INITIALISED;
  lhcb_ctx* c = p->ctx;
  if (!ev || !velo || !so || !lo || ev->n_events < 0 || velo->n_events != ev->n_events || !ev->zone_off || !velo->off ||
      !so->off || !so->state || !so->hits || !so->nx || !so->nuv || !so->status || !lo->off || !lo->seed_idx ||
      !lo->velo_idx || !lo->ut_idx || !lo->n_ut || !lo->qop || !lo->chi2 || !lo->status)
    return LHCB_ERR_BAD_ARGUMENT;
  if (ut && (!ut->off || (!ut->x0 && !ut->strip) || !ut->row)) return LHCB_ERR_BAD_ARGUMENT;   // strip rows, not two floats per hit
  const int n = ev->n_events;
  p->h2d = p->d2h = 0; p->launches = 0;
  so->n = 0; lo->n = 0;
  if (n == 0) { so->off[0] = 0; lo->off[0] = 0; return LHCB_OK; }
  if (n > p->max_events || ev->n_hits > p->max_hits) return LHCB_ERR_CAPACITY;
  const size_t n_velo = velo->off[n];
  const size_t n_ut = ut ? ut->off[(size_t)n * 4] : 0;
  if (n_velo > p->max_velo || n_ut > p->max_ut) return LHCB_ERR_CAPACITY;
  LHCB_CUDA(c, cudaSetDevice(c->device));
  int rc = LHCB_OK;
  cudaError_t ce = cudaSuccess;
  auto H2D = [&](void* d, const void* h, size_t bytes) {
    if (ce != cudaSuccess || !bytes) return;
    p->h2d += bytes;
    ce = cudaMemcpyAsync(d, h, bytes, cudaMemcpyHostToDevice, p->st_in);
  };
  auto D2H = [&](void* h, const void* d, size_t bytes) {
    if (ce != cudaSuccess || !bytes) return;
    p->d2h += bytes;
    ce = cudaMemcpyAsync(h, d, bytes, cudaMemcpyDeviceToHost, p->st_out);
  };
  auto D2H2D = [&](void* h, size_t hpitch, const void* d, size_t dpitch, size_t width, size_t rows) {
    if (ce != cudaSuccess || !width) return;
    p->d2h += width * rows;
    ce = cudaMemcpy2DAsync(h, hpitch, d, dpitch, width, rows, cudaMemcpyDeviceToHost, p->st_out);
  };
  const bool has_pol = ev->polarity != nullptr, has_ut = ut != nullptr, want_par = so->par != nullptr;
  const bool strips = has_ut && ut->strip != nullptr;
  const unsigned flags = (has_pol ? 1u : 0u) | (has_ut ? 2u : 0u) | (want_par ? 4u : 0u) | (c->nn_on ? 8u : 0u) |
                         (c->uv_hough ? 16u : 0u) | (strips ? 32u : 0u);
  // slice table: full slices, the last one cut into halves (1/2, 1/4, 1/4) so that the part of the pipeline that
  // nothing overlaps (kernels and output copies of the final slice) is short
  int ns = 0;
  {
    int e = 0;
    while (n - e > p->slice) { p->e0[ns++] = e; e += p->slice; }
    int rem = n - e;
    for (int piece = 0; piece < 2 && rem >= 512; ++piece) {
      const int half = ((rem / 2) + 63) & ~63;
      p->e0[ns++] = e; e += half; rem -= half;
    }
    p->e0[ns++] = e;
    p->e0[ns] = n;
  }
  // ---- all input copies on the copy-in stream.  The small arrays (offsets, polarities, VELO states: a few per
  // cent of the bytes) go first, each as ONE copy for the whole batch: a copy costs a few microseconds whatever
  // its size, and a dozen of them per slice add up to a millisecond per batch.  The hits then follow slice by
  // slice.
  {
    const size_t n_velo_all = velo->off[n];
    H2D(p->zone_off, ev->zone_off, ((size_t)n * 24 + 1) * 4);
    if (has_pol) H2D(p->pol, ev->polarity, (size_t)n);
    H2D(p->velo_off, velo->off, ((size_t)n + 1) * 4);
    H2D(p->vx, velo->x, n_velo_all * 4);
    H2D(p->vy, velo->y, n_velo_all * 4);
    H2D(p->vtx, velo->tx, n_velo_all * 4);
    H2D(p->vty, velo->ty, n_velo_all * 4);
    if (has_ut) H2D(p->ut_off, ut->off, ((size_t)n * 4 + 1) * 4);
  }
  for (int k = 0; k < ns && ce == cudaSuccess; ++k) {
    const int e0 = p->e0[k], ne = p->e0[k + 1] - e0;
    const size_t z0 = (size_t)e0 * 24, z1 = (size_t)(e0 + ne) * 24;
    const size_t h0 = ev->zone_off[z0], h1 = ev->zone_off[z1];
    H2D(p->hit_x + h0, ev->hit_x + h0, (h1 - h0) * 4);
    if (has_ut) {
      const size_t u0 = ut->off[(size_t)e0 * 4], u1 = ut->off[(size_t)(e0 + ne) * 4];
      if (strips) H2D(p->ustrip + u0, ut->strip + u0, (u1 - u0) * 2);
      else H2D(p->ux + u0, ut->x0 + u0, (u1 - u0) * 4);
      H2D(p->urow + u0, ut->row + u0, u1 - u0);
    }
    if (ce == cudaSuccess) ce = cudaEventRecord(p->ev_in[k], p->st_in);
  }
  // ---- kernels: one graph per slice on the compute stream
  if (ce == cudaSuccess) ce = cudaMemsetAsync(p->totals, 0, 8, p->st_k);
  for (int k = 0; k < ns && ce == cudaSuccess && rc == LHCB_OK; ++k) {
    const int e0 = p->e0[k], ne = p->e0[k + 1] - e0;
    lhcb_pipeline::Graph& G = p->graphs[k];
    if (!G.exec || G.e0 != e0 || G.ne != ne || G.flags != flags) {
      if (G.exec) { cudaGraphExecDestroy(G.exec); G.exec = nullptr; }
      cudaGraph_t graph = nullptr;
      ce = cudaStreamBeginCapture(p->st_k, cudaStreamCaptureModeThreadLocal);
      if (ce != cudaSuccess) break;
      rc = enqueue_slice(p, k, e0, ne, has_ut, has_pol, want_par, strips, &G.launches);
      const cudaError_t ec = cudaStreamEndCapture(p->st_k, &graph);
      if (rc != LHCB_OK) { if (graph) cudaGraphDestroy(graph); break; }
      ce = ec;
      if (ce == cudaSuccess) ce = cudaGraphInstantiate(&G.exec, graph, 0);
      if (graph) cudaGraphDestroy(graph);
      if (ce != cudaSuccess) { G.exec = nullptr; break; }
      G.e0 = e0; G.ne = ne; G.flags = flags;
    }
    ce = cudaStreamWaitEvent(p->st_k, p->ev_in[k], 0);
    if (ce == cudaSuccess) ce = cudaGraphLaunch(G.exec, p->st_k);
    if (ce == cudaSuccess) ce = cudaEventRecord(p->ev_k[k], p->st_k);
    p->launches += G.launches;                               // (strip decoding,) order, seeding, matching, scan, gather: counted at capture
  }
  // ---- outputs: as soon as a slice's totals are known, exactly its entries are copied
  uint32_t seeds_end = 0, long_end = 0;
  for (int k = 0; k < ns && ce == cudaSuccess && rc == LHCB_OK; ++k) {
    const int e0 = p->e0[k], ne = p->e0[k + 1] - e0;
    ce = cudaEventSynchronize(p->ev_k[k]);
      if (ce != cudaSuccess) break;
    const uint32_t sb = p->h_totals[k * 4], se = p->h_totals[k * 4 + 1], lb = p->h_totals[k * 4 + 2], le = p->h_totals[k * 4 + 3];
    if (se > p->cap_s || le > p->cap_l || se > so->cap || le > lo->cap) { rc = LHCB_ERR_CAPACITY; break; }
    seeds_end = se; long_end = le;
    const size_t CS = p->cap_s, CL = p->cap_l, hs = so->cap, hl = lo->cap, nsd = se - sb, nl = le - lb;
    D2H2D(so->state + sb, hs * 4, p->d_state + sb, CS * 4, nsd * 4, 5);
    D2H2D(so->hits + sb, hs * 2, p->d_hits + sb, CS * 2, nsd * 2, 12);
    if (want_par) D2H2D(so->par + sb, hs * 4, p->d_par + sb, CS * 4, nsd * 4, 7);
    D2H(so->nx + sb, p->d_nx + sb, nsd);
    D2H(so->nuv + sb, p->d_nuv + sb, nsd);
    D2H(lo->seed_idx + lb, p->d_seed + lb, nl * 4);
    D2H(lo->velo_idx + lb, p->d_velo + lb, nl * 4);
    D2H2D(lo->ut_idx + lb, hl * 4, p->d_ut + lb, CL * 4, nl * 4, 4);
    D2H(lo->n_ut + lb, p->d_nut + lb, nl);
    D2H(lo->qop + lb, p->d_qop + lb, nl * 4);
    D2H(lo->chi2 + lb, p->d_chi2 + lb, nl * 4);
  }
  // offsets and status words of the whole batch: one copy each (the last slice's kernels have finished)
  if (ce == cudaSuccess && rc == LHCB_OK) {
    D2H(so->off, p->d_s_off, ((size_t)n * 2 + 1) * 4);
    D2H(so->status, p->d_s_status, (size_t)n * 8);
    D2H(lo->off, p->d_l_off, ((size_t)n + 1) * 4);
    D2H(lo->status, p->d_l_status, (size_t)n * 4);
  }
  // every stream is drained before returning, whatever happened: no copy is left in flight on the caller's buffers
  const cudaError_t e1 = cudaStreamSynchronize(p->st_in), e2 = cudaStreamSynchronize(p->st_k), e3 = cudaStreamSynchronize(p->st_out);
  if (ce == cudaSuccess) ce = e1 != cudaSuccess ? e1 : (e2 != cudaSuccess ? e2 : e3);
  if (rc != LHCB_OK) return rc;
  if (ce != cudaSuccess) return cuda_fail(c, ce);
  so->n = seeds_end; lo->n = long_end;
  return LHCB_OK;
}

int lhcb_pipeline_last_bytes(const lhcb_pipeline* p, uint64_t* h2d, uint64_t* d2h) {
  if (!p) return LHCB_ERR_NOT_INITIALISED;
  if (h2d) *h2d = p->h2d;
  if (d2h) *d2h = p->d2h;
  return p->launches;
}

}  // extern "C"
