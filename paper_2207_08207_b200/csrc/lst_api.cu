// lst_api.cu -- host side of liblst.so: the C-ABI of include/lst.h, the arena and the slots.
//
// Runtime design:
//  * lst_create allocates once: the arena (every slot's input staging, hit store, object store, CSR offsets and
//    scratch) and five small geometry / map tables; per event nothing is allocated or freed, and a slot recycles
//    itself inside the a0 kernels (bin counters cleared by the block that scans them, a fresh header written by the
//    same block, look-back words cleared by the scatter kernel): no reset launch.
//  * lst_load_event / lst_run* only enqueue work on the caller's stream; sizes that are only
//    known on the device (object counts) never come back to the host between stages: grids
//    are fixed by the geometry / capacities and kernels read the counts from the slot header.
//    The enqueue sequence is therefore capturable into a CUDA graph by the caller.
//  * a batch of slots runs through ONE launch per kernel (grid.y = batch index).
#include <cuda_runtime.h>

#include <atomic>
#include <cstdlib>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

#include "../../include/lst.h"
#include "lst_device.cuh"

using namespace lst;

static_assert((int)LST_MD == (int)LST_MD_ && (int)LST_SEG == (int)LST_SEG_ && (int)LST_T3 == (int)LST_T3_ &&
                  (int)LST_T5 == (int)LST_T5_ && (int)LST_CLEAN == (int)LST_CLEAN_ && (int)LST_PIXEL == (int)LST_PIXEL_, "stage ids");

static_assert(sizeof(SlotHeader) == 424, "bench.py HEADER_BYTES counts the header lst_sync_batch reads back");

namespace {

struct SlotHost {
  bool loaded = false, synced = false;
  int stages_run = 0;         // stages a1 .. run in order since the load: objects of class k are valid iff stages_run > k
  int n_hits_in = 0;
  SlotHeader* hdr = nullptr;  // pinned host copy of the device header
  bool seeds_loaded = false, pixel_run = false;   // [P]: lst_load_seeds since the last lst_load_event; LST_PIXEL since then
  int n_seeds_in = 0;
  int seed_owner = -1;        // >= 0: the seed binning of this slot runs on a side stream and has not been joined yet; the slot whose seed_done event marks its end
  cudaEvent_t seed_fork = nullptr, seed_done = nullptr;
  cudaEvent_t ev[22] = {};    // timing mode: ev[0..3] around the 3 a0 kernels, ev[4 + 2 s], ev[5 + 2 s] around stage s, ev[12..16] around the 4 cleaning steps, ev[17..18] around k_seed_bin, ev[19..21] around the two link kernels
  bool ev_bin = false, ev_stage[5] = {false, false, false, false, false}, ev_seed = false, ev_pix = false;
};

}  // namespace

struct lst_ctx {
  lst_config cfg;
  Params P;  // first_slot filled per call
  int device = 0;
  signed char* d_layer = nullptr;
  float2* d_mod_cs = nullptr;
  int* d_map_offsets = nullptr;
  int* d_map_targets = nullptr;
  float* d_map_dphi = nullptr;
  int* d_map_targets_asc = nullptr;   // the rows as the caller gave them (ascending target), with their azimuth offsets
  float* d_map_dphi_asc = nullptr;
  char* arena = nullptr;
  size_t arena_bytes = 0;
  std::vector<SlotHost> slots;
  SlotHeader* pinned = nullptr;
  // Stage-in kernels (k_bin_count reading pinned host memory) run on the library's own high-priority stream,
  // forked from and joined to the caller's stream by events: like copies on a copy engine they are served one
  // after the other at full link speed, and the next batch's stage-in overlaps this batch's stage kernels.
  static constexpr int kStageEvents = 32;
  cudaStream_t stage_stream = nullptr;
  cudaEvent_t stage_ev[kStageEvents] = {};
  unsigned stage_next = 0;
  std::mutex stage_mu;
  // [P] The seed binning (one latency-bound block per event) depends on nothing but the slot's fresh header, and only the link
  // kernels need it: lst_load_seeds forks it onto one of these streams so that it runs beside a0 .. a4 of the same batch, and
  // LST_PIXEL (or the next load / sync of the slot) joins it.
  static constexpr int kSeedStreams = 4;
  cudaStream_t seed_stream[kSeedStreams] = {};
  std::atomic<long long> launches{0};
  std::atomic<int> last_cuda{0};
};

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int fail_cuda(lst_ctx* c, cudaError_t e) {
  if (c) c->last_cuda.store((int)e);
  return LST_ERR_CUDA;
}
#define LST_CUDA(ctx, call)                              \
  do {                                                   \
    cudaError_t e__ = (call);                            \
    if (e__ != cudaSuccess) return fail_cuda(ctx, e__);  \
  } while (0)

Layout make_layout(const lst_config& cfg, int n_modules) {
  Layout L{};
  L.n_modules = n_modules;
  L.n_bins = 2 * n_modules;
  L.cap_hits = cfg.cap_hits; L.cap_md = cfg.cap_md; L.cap_seg = cfg.cap_seg; L.cap_t3 = cfg.cap_t3; L.cap_t5 = cfg.cap_t5;
  L.cap_seeds = cfg.cap_seeds; L.cap_pix[0] = cfg.cap_pt3; L.cap_pix[1] = cfg.cap_pt5;
  L.n_chunk_pix[0] = (cfg.cap_t3 + kChunk - 1) / kChunk; L.n_chunk_pix[1] = (cfg.cap_t5 + kChunk - 1) / kChunk;
  const int owner_cap[4] = {cfg.cap_hits, cfg.cap_md, cfg.cap_seg, cfg.cap_t3};
  for (int k = 0; k < 4; ++k) L.n_chunk[k] = (owner_cap[k] + kChunk - 1) / kChunk;
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
  L.hdr = take(sizeof(SlotHeader));
  L.bin_cnt = take(sizeof(int) * (size_t)(L.n_bins + 1));
  L.bin_start = take(sizeof(int) * (size_t)(L.n_bins + 1));
  for (int k = 0; k < 4; ++k) L.lb[k] = take(8 * (size_t)(L.n_chunk[k] + 1));
  L.lb_bytes = off - L.lb[0];
  const size_t nh = (size_t)cfg.cap_hits, nm = (size_t)cfg.cap_md, ns = (size_t)cfg.cap_seg, n3 = (size_t)cfg.cap_t3, n5 = (size_t)cfg.cap_t5;
  L.in_x = take(4 * nh); L.in_y = take(4 * nh); L.in_z = take(4 * nh); L.in_module = take(4 * nh); L.in_side = take(nh);
  L.rec4 = take(16 * nh); L.recb = take(8 * nh); L.reck = take(4 * nh);
  L.tmp_ki = take(8 * nh); L.tmp_bin = take(4 * nh);
  L.hit4 = take(16 * nh); L.hit_key = take(4 * nh); L.hit_orig = take(4 * nh); L.hit_module = take(4 * nh);
  L.md_start = take(4 * (size_t)(n_modules + 1)); L.mod_info = take(16 * (size_t)n_modules);
  L.md_anchor = take(16 * nm); L.md_aux = take(8 * nm); L.md_key = take(4 * nm); L.md_hits = take(8 * nm);
  L.md_out = take(8 * nm); L.md_module = take(4 * nm);
  L.seg_start = take(4 * (nm + 1));
  L.seg_md = take(8 * ns); L.seg_f = take(16 * ns);
  L.t3_start = take(4 * (ns + 1));
  L.t3_pack = take(16 * n3); L.t3_seg = take(8 * n3); L.t3_chi2 = take(4 * n3);
  L.t5_start = take(4 * (n3 + 1));
  L.t5_md = take(20 * n5); L.t5_t3 = take(8 * n5); L.t5_f = take(20 * n5); L.t5_kfit = take(4 * n5);
  L.t5_hits = take(40 * n5); L.t5_score = take(4 * n5); L.t5_keep = take(n5); L.tc_list = take(4 * n5);
  L.inc_start = take(4 * (nm + 8)); L.inc_cur = take(4 * (nm + 8)); L.inc_list = take(40 * n5);
  {  // [P]
    const size_t nsd = (size_t)cfg.cap_seeds;
    L.seed_in = take(20 * nsd);
    L.seed_rec4 = take(16 * nsd * kSeedBands); L.seed_rec2 = take(8 * nsd * kSeedBands);   // a seed is filed once per curvature band it can match
    L.seed_bin_start = take(4 * (size_t)(kSeedBins + 3));
    for (int k = 0; k < 2; ++k) L.lb_pix[k] = take(8 * (size_t)(L.n_chunk_pix[k] + 1));
    L.lb_pix_bytes = off - L.lb_pix[0];
    const size_t nobj[2] = {n3, n5};
    for (int k = 0; k < 2; ++k) {
      L.pix_start[k] = take(4 * (nobj[k] + 1));
      L.pix_link[k] = take(8 * (size_t)L.cap_pix[k]);
      L.pix_f[k] = take(12 * (size_t)L.cap_pix[k]);
    }
  }
  size_t scr = 16 * nm;   // one gathered table at a time: hit-index tuples (8 / 16 / 24 / 40 B) or packed values (16 / 16 / 8 / 20 B)
  if (16 * ns > scr) scr = 16 * ns;
  if (24 * n3 > scr) scr = 24 * n3;
  if (40 * n5 > scr) scr = 40 * n5;
  L.scratch = take(scr);
  L.slot_bytes = align_up(off, 4096);
  return L;
}

// Device-visible alias of a pinned (page-locked, mapped) host pointer, or nullptr for pageable memory.
const void* mapped_alias(const void* p) {
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return nullptr; }
  return a.type == cudaMemoryTypeHost ? a.devicePointer : nullptr;
}
// True (and the pointers replaced by their device-visible aliases) if all five arrays are pinned host memory.
bool mapped_host(HitInput& in) {
  const void* p[5] = {mapped_alias(in.x), mapped_alias(in.y), mapped_alias(in.z), mapped_alias(in.module), mapped_alias(in.side)};
  for (const void* q : p)
    if (!q) return false;
  in.x = static_cast<const float*>(p[0]); in.y = static_cast<const float*>(p[1]); in.z = static_cast<const float*>(p[2]);
  in.module = static_cast<const int*>(p[3]); in.side = static_cast<const unsigned char*>(p[4]);
  return true;
}

bool valid_slot(const lst_ctx* c, int slot) { return c && slot >= 0 && slot < (int)c->slots.size(); }

// Makes `s` wait for the seed binning of slots first .. first + n - 1 that still runs on a side stream (one wait per batch).
cudaError_t join_seeds(lst_ctx* c, int first, int n, cudaStream_t s) {
  int last_owner = -1;
  for (int k = first; k < first + n; ++k) {
    SlotHost& sh = c->slots[k];
    if (sh.seed_owner < 0) continue;
    if (sh.seed_owner != last_owner) {
      const cudaError_t e = cudaStreamWaitEvent(s, c->slots[sh.seed_owner].seed_done, 0);
      if (e != cudaSuccess) return e;
      last_owner = sh.seed_owner;
    }
    sh.seed_owner = -1;
  }
  return cudaSuccess;
}

void copy_cuts(Cuts& d, const lst_config& s) {
  d.half_kappa_max = s.half_kappa_max; d.z_lum = s.z_lum;
  for (int i = 0; i < 6; ++i) {
    d.md_cos_eps[i] = s.md_cos_eps[i]; d.md_sin_eps[i] = s.md_sin_eps[i]; d.md_dz_res[i] = s.md_dz_res[i];
    d.md_eps[i] = s.md_eps[i]; d.sigma_z2[i] = s.sigma_z2[i]; d.inv_sigma_z2[i] = s.inv_sigma_z2[i];
  }
  d.seg_cos_eps = s.seg_cos_eps; d.seg_sin_eps = s.seg_sin_eps;
  for (int i = 0; i < 5; ++i) d.seg_z0_max[i] = s.seg_z0_max[i];
  d.t3_kappa_max = s.t3_kappa_max;
  for (int i = 0; i < 4; ++i) d.t3_chi2rz_max[i] = s.t3_chi2rz_max[i];
  d.t5_dkappa_max = s.t5_dkappa_max;
  for (int i = 0; i < 2; ++i) d.t5_chi2rz_max[i] = s.t5_chi2rz_max[i];
  d.t5_chi2xy_max = s.t5_chi2xy_max; d.t5_sigma_xy2_scaled = s.t5_sigma_xy2_scaled; d.t5_kappa_max = s.t5_kappa_max;
  for (int i = 0; i < 2; ++i) { d.pix_dkappa_max[i] = s.pix_dkappa_max[i]; d.pix_chi2xy_max[i] = s.pix_chi2xy_max[i]; d.pix_chi2rz_max[i] = s.pix_chi2rz_max[i]; }
  for (int i = 0; i < 6; ++i) { d.pix_inv_var_xy[i] = s.pix_inv_var_xy[i]; d.pix_inv_var_rz[i] = s.pix_inv_var_rz[i]; }
}

}  // namespace

extern "C" {

int lst_default_config(lst_config* c) {
  if (!c) return LST_ERR_ARG;
  std::memset(c, 0, sizeof(*c));
  // DESIGN.md section 1, "Constants", typed from the table
  c->half_kappa_max = 0.00712007098f;
  c->z_lum = 15.0f;
  for (int l = 0; l < LST_N_LAYERS; ++l) {
    const bool ps = l < 3;
    c->md_cos_eps[l] = ps ? 0.99840045f : 0.995777965f;
    c->md_sin_eps[l] = ps ? 0.056538377f : 0.0917944759f;
    c->md_eps[l] = ps ? 0.0565685406f : 0.091923885f;
    c->md_dz_res[l] = ps ? 0.243244737f : 7.91959572f;
    c->sigma_z2[l] = ps ? 0.001849f : 1.96f;
    c->inv_sigma_z2[l] = ps ? 540.832886f : 0.510204077f;
  }
  c->seg_cos_eps = 0.999997973f;
  c->seg_sin_eps = 0.0019999987f;
  const float zseg[5] = {20.0f, 20.0f, 40.0f, 90.0f, 90.0f};
  for (int l = 0; l < 5; ++l) c->seg_z0_max[l] = zseg[l];
  c->t3_kappa_max = 0.0149521492f;
  const float t3c[4] = {100.0f, 30.0f, 25.0f, 25.0f};
  for (int l = 0; l < 4; ++l) c->t3_chi2rz_max[l] = t3c[l];
  c->t5_dkappa_max = 0.000284802838f;
  c->t5_chi2rz_max[0] = 110.0f;
  c->t5_chi2rz_max[1] = 150.0f;
  c->t5_chi2xy_max = 35.0f;
  c->t5_sigma_xy2_scaled = 6.6015625e-09f;
  c->t5_kappa_max = 0.0149521492f;
  c->pix_dkappa_max[0] = 0.0008f; c->pix_dkappa_max[1] = 0.0007f;
  const float pvx[6] = {809.479f, 187.19363f, 51.984085f, 16.645065f, 6.149085f, 2.8425808f};
  const float pvz[6] = {229.09508f, 136.11072f, 79.544624f, 0.50524855f, 0.5020406f, 0.4982422f};
  for (int l = 0; l < LST_N_LAYERS; ++l) { c->pix_inv_var_xy[l] = pvx[l]; c->pix_inv_var_rz[l] = pvz[l]; }
  c->pix_chi2xy_max[0] = 85.0f; c->pix_chi2xy_max[1] = 145.0f;
  c->pix_chi2rz_max[0] = 25.0f; c->pix_chi2rz_max[1] = 35.0f;
  c->device = 0;
  c->n_slots = 4;
  c->cap_hits = 192 * 1024;
  c->cap_md = 96 * 1024;
  c->cap_seg = 256 * 1024;
  c->cap_t3 = 384 * 1024;
  c->cap_t5 = 128 * 1024;
  c->timing = 0;
  c->t5_dup_min_shared = 7;
  c->store_half = 0;
  c->launches_in_flight = 0;
  c->cap_seeds = 16 * 1024;
  c->cap_pt3 = 64 * 1024;
  c->cap_pt5 = 64 * 1024;
  return LST_OK;
}

int lst_create(const lst_geometry* g, const lst_module_map* m, const lst_config* cfg_in, lst_ctx** out) {
  if (!g || !m || !out) return LST_ERR_ARG;
  *out = nullptr;
  lst_config cfg;
  if (cfg_in) cfg = *cfg_in; else lst_default_config(&cfg);
  const int n = g->n_modules;
  if (n <= 0 || n > (1 << 24) || m->n_modules != n || !g->layer || !g->phi || !m->row_offsets) return LST_ERR_ARG;
  /* object indices are packed into 26 bits, module ids into 24 bits by the stage kernels */
  if (cfg.cap_hits > kMaxCap || cfg.cap_md > kMaxCap || cfg.cap_seg > kMaxCap || cfg.cap_t3 > kMaxCap || cfg.cap_t5 > kMaxCap) return LST_ERR_ARG;
  /* [D]: partners are found through a common mini-doublet, which two quintuplets sharing >= 6 of their 10 hits always
     have (five common layers with one common hit each give at most 5): smaller thresholds are refused, not approximated */
  if (cfg.t5_dup_min_shared < 6 || cfg.t5_dup_min_shared > 10) return LST_ERR_ARG;
  if (cfg.launches_in_flight < 0) return LST_ERR_ARG;
  if (cfg.n_slots < 1 || cfg.cap_hits < 1 || cfg.cap_md < 1 || cfg.cap_seg < 1 || cfg.cap_t3 < 1 || cfg.cap_t5 < 1) return LST_ERR_ARG;
  if (cfg.cap_seeds < 1 || cfg.cap_pt3 < 1 || cfg.cap_pt5 < 1 || cfg.cap_seeds > kMaxCap || cfg.cap_pt3 > kMaxCap || cfg.cap_pt5 > kMaxCap) return LST_ERR_ARG;
  for (int i = 0; i < n; ++i)
    if (g->layer[i] < 0 || g->layer[i] >= LST_N_LAYERS) return LST_ERR_ARG;
  if (m->row_offsets[0] != 0) return LST_ERR_ARG;
  for (int i = 0; i < n; ++i)
    if (m->row_offsets[i + 1] < m->row_offsets[i]) return LST_ERR_ARG;
  if (m->row_offsets[n] > 0 && !m->targets) return LST_ERR_ARG;
  // rows strictly ascending, targets in the next layer, at most kMaxRow connections per module
  const double kPi = 3.14159265358979323846;
  const int n_conn = m->row_offsets[n];
  std::vector<float> map_dphi((size_t)n_conn + 1, 0.0f);
  std::vector<int> map_tgt((size_t)n_conn + 1, 0);   // rows re-ordered by (azimuth offset, target) for the segment kernel
  std::vector<float> map_dphi_asc((size_t)n_conn + 1, 0.0f);   // offsets in the caller's order (ascending target)
  std::vector<float2> mod_cs(n);
  for (int a = 0; a < n; ++a) {
    if (!std::isfinite(g->phi[a])) return LST_ERR_ARG;
    mod_cs[a] = make_float2((float)std::cos((double)g->phi[a]), (float)std::sin((double)g->phi[a]));
    if (m->row_offsets[a + 1] - m->row_offsets[a] > kMaxRow) return LST_ERR_ARG;
    for (int k = m->row_offsets[a]; k < m->row_offsets[a + 1]; ++k) {
      const int t = m->targets[k];
      if (t < 0 || t >= n || g->layer[t] != g->layer[a] + 1) return LST_ERR_ARG;
      if (k > m->row_offsets[a] && t <= m->targets[k - 1]) return LST_ERR_ARG;
      if (!std::isfinite(g->phi[t])) return LST_ERR_ARG;
      double d = std::fmod((double)g->phi[a] - (double)g->phi[t], 2.0 * kPi);  // into (-pi, pi]
      if (d > kPi) d -= 2.0 * kPi;
      if (d <= -kPi) d += 2.0 * kPi;
      map_dphi[k] = (float)d;
      map_dphi_asc[k] = (float)d;
      map_tgt[k] = t;
    }
    // insertion sort of the row (at most kMaxRow entries) by (azimuth offset, target)
    for (int k = m->row_offsets[a] + 1; k < m->row_offsets[a + 1]; ++k) {
      const float d = map_dphi[k];
      const int t = map_tgt[k];
      int j = k - 1;
      for (; j >= m->row_offsets[a] && (map_dphi[j] > d || (map_dphi[j] == d && map_tgt[j] > t)); --j) {
        map_dphi[j + 1] = map_dphi[j];
        map_tgt[j + 1] = map_tgt[j];
      }
      map_dphi[j + 1] = d;
      map_tgt[j + 1] = t;
    }
  }

  lst_ctx* c = new (std::nothrow) lst_ctx();
  if (!c) return LST_ERR_NOMEM;
  c->cfg = cfg;
  c->device = cfg.device;
  auto bail = [&](int status, cudaError_t e) {
    if (status == LST_ERR_CUDA) c->last_cuda.store((int)e);
    lst_destroy(c);
    return status;
  };
  cudaError_t e;
  if ((e = cudaSetDevice(cfg.device)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  const Layout L = make_layout(cfg, n);
  c->arena_bytes = L.slot_bytes * (size_t)cfg.n_slots;
  if ((e = cudaMalloc(&c->d_layer, n)) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->d_mod_cs, sizeof(float2) * n)) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->d_map_offsets, sizeof(int) * (n + 1))) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->d_map_targets, sizeof(int) * ((size_t)n_conn + 1))) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->d_map_dphi, sizeof(float) * ((size_t)n_conn + 1))) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->d_map_targets_asc, sizeof(int) * ((size_t)n_conn + 1))) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->d_map_dphi_asc, sizeof(float) * ((size_t)n_conn + 1))) != cudaSuccess) return bail(LST_ERR_NOMEM, e);
  if ((e = cudaMalloc(&c->arena, c->arena_bytes)) != cudaSuccess) { cudaGetLastError(); return bail(LST_ERR_NOMEM, e); }
  if ((e = cudaMemcpy(c->d_layer, g->layer, n, cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if ((e = cudaMemcpy(c->d_mod_cs, mod_cs.data(), sizeof(float2) * n, cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if ((e = cudaMemcpy(c->d_map_offsets, m->row_offsets, sizeof(int) * (n + 1), cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if (n_conn > 0 && (e = cudaMemcpy(c->d_map_targets, map_tgt.data(), sizeof(int) * (size_t)n_conn, cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if (n_conn > 0 && (e = cudaMemcpy(c->d_map_dphi, map_dphi.data(), sizeof(float) * (size_t)n_conn, cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if (n_conn > 0 && (e = cudaMemcpy(c->d_map_targets_asc, m->targets, sizeof(int) * (size_t)n_conn, cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if (n_conn > 0 && (e = cudaMemcpy(c->d_map_dphi_asc, map_dphi_asc.data(), sizeof(float) * (size_t)n_conn, cudaMemcpyHostToDevice)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if ((e = cudaMemset(c->arena, 0, c->arena_bytes)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  if ((e = cudaMallocHost(&c->pinned, sizeof(SlotHeader) * (size_t)cfg.n_slots)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  std::memset(c->pinned, 0, sizeof(SlotHeader) * (size_t)cfg.n_slots);
  {
    int lo = 0, hi = 0;
    if ((e = cudaDeviceGetStreamPriorityRange(&lo, &hi)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
    if ((e = cudaStreamCreateWithPriority(&c->stage_stream, cudaStreamNonBlocking, hi)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
    for (auto& ev : c->stage_ev)
      if ((e = cudaEventCreateWithFlags(&ev, cudaEventDisableTiming)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  }
  for (auto& st : c->seed_stream)
    if ((e = cudaStreamCreateWithFlags(&st, cudaStreamNonBlocking)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  c->slots.resize(cfg.n_slots);
  for (int s = 0; s < cfg.n_slots; ++s) {
    c->slots[s].hdr = c->pinned + s;
    if ((e = cudaEventCreateWithFlags(&c->slots[s].seed_fork, cudaEventDisableTiming)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
    if ((e = cudaEventCreateWithFlags(&c->slots[s].seed_done, cudaEventDisableTiming)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
    if (cfg.timing)
      for (auto& ev : c->slots[s].ev)
        if ((e = cudaEventCreate(&ev)) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  }
  c->P.arena = c->arena;
  c->P.slot_stride = L.slot_bytes;
  c->P.L = L;
  copy_cuts(c->P.cuts, cfg);
  c->P.mod_layer = c->d_layer;
  c->P.mod_cs = c->d_mod_cs;
  c->P.map_offsets = c->d_map_offsets;
  c->P.map_targets = c->d_map_targets;
  c->P.map_dphi = c->d_map_dphi;
  c->P.map_targets_asc = c->d_map_targets_asc;
  c->P.map_dphi_asc = c->d_map_dphi_asc;
  c->P.first_slot = 0;
  c->P.dup_min_shared = cfg.t5_dup_min_shared;
  c->P.store_half = cfg.store_half != 0;
  c->P.four_launches = cfg.launches_in_flight >= 4;
  for (int k = 0; k < 3; ++k) {  // are the modules of layers <= 1 / <= 3 / <= 4 a prefix of the module ids?
    const int max_layer = k == 0 ? 1 : k == 1 ? 3 : 4;
    int live = 0;
    while (live < n && g->layer[live] <= max_layer) ++live;
    bool prefix = true;
    for (int i = live; i < n; ++i) prefix = prefix && g->layer[i] > max_layer;
    c->P.live_modules[k] = prefix ? live : n;
  }
  if ((e = cudaDeviceSynchronize()) != cudaSuccess) return bail(LST_ERR_CUDA, e);
  *out = c;
  return LST_OK;
}

int lst_destroy(lst_ctx* c) {
  if (!c) return LST_ERR_ARG;
  cudaSetDevice(c->device);
  for (auto& s : c->slots) {
    for (auto& ev : s.ev)
      if (ev) cudaEventDestroy(ev);
    if (s.seed_fork) cudaEventDestroy(s.seed_fork);
    if (s.seed_done) cudaEventDestroy(s.seed_done);
  }
  for (auto& st : c->seed_stream)
    if (st) cudaStreamDestroy(st);
  for (auto& ev : c->stage_ev)
    if (ev) cudaEventDestroy(ev);
  if (c->stage_stream) cudaStreamDestroy(c->stage_stream);
  if (c->pinned) cudaFreeHost(c->pinned);
  if (c->arena) cudaFree(c->arena);
  if (c->d_map_dphi) cudaFree(c->d_map_dphi);
  if (c->d_map_dphi_asc) cudaFree(c->d_map_dphi_asc);
  if (c->d_map_targets_asc) cudaFree(c->d_map_targets_asc);
  if (c->d_map_targets) cudaFree(c->d_map_targets);
  if (c->d_map_offsets) cudaFree(c->d_map_offsets);
  if (c->d_mod_cs) cudaFree(c->d_mod_cs);
  if (c->d_layer) cudaFree(c->d_layer);
  delete c;
  return LST_OK;
}

int lst_load_events(lst_ctx* c, int first, int n_ev, const lst_hits* hits, void* stream) {
  if (!c || n_ev < 1 || !valid_slot(c, first) || !valid_slot(c, first + n_ev - 1) || !hits) return LST_ERR_ARG;
  for (int b = 0; b < n_ev; ++b) {
    const lst_hits* h = hits + b;
    if (h->n < 0) return LST_ERR_ARG;
    if (h->n > 0 && (!h->x || !h->y || !h->z || !h->module || !h->side)) return LST_ERR_ARG;
    if (h->n > c->cfg.cap_hits) return LST_ERR_OVERFLOW;
  }
  cudaStream_t s = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  LST_CUDA(c, join_seeds(c, first, n_ev, s));   // a seed binning still in flight on these slots must not meet the new header
  const Layout& L = c->P.L;
  for (int b0 = 0; b0 < n_ev; b0 += kMaxBatch) {
    const int nb = n_ev - b0 < kMaxBatch ? n_ev - b0 : kMaxBatch;
    HitBatch src;
    std::memset(&src, 0, sizeof(src));
    for (int b = 0; b < nb; ++b) {
      const int slot = first + b0 + b;
      const lst_hits* h = hits + b0 + b;
      SlotHost& sh = c->slots[slot];
      sh.loaded = sh.synced = false;
      sh.stages_run = 0;
      sh.n_hits_in = h->n;
      sh.ev_bin = false;
      for (bool& f : sh.ev_stage) f = false;
      sh.seeds_loaded = sh.pixel_run = sh.ev_seed = sh.ev_pix = false;
      char* base = c->arena + (size_t)slot * c->P.slot_stride;
      HitInput in{h->x, h->y, h->z, h->module, h->side, h->n, 0};
      const HitInput staged{reinterpret_cast<const float*>(base + L.in_x), reinterpret_cast<const float*>(base + L.in_y),
                            reinterpret_cast<const float*>(base + L.in_z), reinterpret_cast<const int*>(base + L.in_module),
                            reinterpret_cast<const unsigned char*>(base + L.in_side), h->n, 0};
      // "packed" host layout: the five arrays back to back in ONE block, each starting on a 256-byte boundary
      // (x at p, y at p + A, z at p + 2 A, module at p + 3 A, side at p + 4 A, A = 4 n rounded up to 256)
      const size_t A = align_up(4 * (size_t)h->n, 256);
      const char* px = reinterpret_cast<const char*>(h->x);
      const bool packed = !h->on_device && h->n > 0 && reinterpret_cast<const char*>(h->y) == px + A &&
                          reinterpret_cast<const char*>(h->z) == px + 2 * A && reinterpret_cast<const char*>(h->module) == px + 3 * A &&
                          reinterpret_cast<const char*>(h->side) == px + 4 * A;
      if (h->on_device || h->n == 0) {
        src.ev[b] = in;
      } else if (packed) {
        // one copy-engine transfer of the whole event (1.3 MB at PU200 density runs at link speed, five 300 kB ones do
        // not), into the same layout in the slot's copy area; no SM involved, full duplex with the result copies
        char* d = base + L.in_x;
        LST_CUDA(c, cudaMemcpyAsync(d, px, 4 * A + (size_t)h->n, cudaMemcpyHostToDevice, s));
        src.ev[b] = HitInput{reinterpret_cast<const float*>(d), reinterpret_cast<const float*>(d + A),
                             reinterpret_cast<const float*>(d + 2 * A), reinterpret_cast<const int*>(d + 3 * A),
                             reinterpret_cast<const unsigned char*>(d + 4 * A), h->n, 0};
      } else if (mapped_host(in)) {
        // pinned host arrays: k_bin_count reads them over PCIe (one coalesced pass); nothing else ever reads them
        in.stage = 1;
        src.ev[b] = in;
      } else {
        // pageable host arrays: the driver stages the copies
        const size_t n = (size_t)h->n;
        LST_CUDA(c, cudaMemcpyAsync(base + L.in_x, h->x, 4 * n, cudaMemcpyHostToDevice, s));
        LST_CUDA(c, cudaMemcpyAsync(base + L.in_y, h->y, 4 * n, cudaMemcpyHostToDevice, s));
        LST_CUDA(c, cudaMemcpyAsync(base + L.in_z, h->z, 4 * n, cudaMemcpyHostToDevice, s));
        LST_CUDA(c, cudaMemcpyAsync(base + L.in_module, h->module, 4 * n, cudaMemcpyHostToDevice, s));
        LST_CUDA(c, cudaMemcpyAsync(base + L.in_side, h->side, n, cudaMemcpyHostToDevice, s));
        src.ev[b] = staged;
      }
    }
    SlotHost& sh0 = c->slots[first + b0];
    Params P = c->P;
    P.first_slot = first + b0;
    bool staged = false;
    for (int b = 0; b < nb; ++b) staged = staged || src.ev[b].stage;
    if (staged) {
      std::lock_guard<std::mutex> lock(c->stage_mu);
      StageIn st{c->stage_stream, c->stage_ev[c->stage_next % lst_ctx::kStageEvents], c->stage_ev[(c->stage_next + 1) % lst_ctx::kStageEvents]};
      c->stage_next += 2;
      c->launches += launch_bin(P, src, nb, s, c->cfg.timing ? sh0.ev : nullptr, &st);
    } else {
      c->launches += launch_bin(P, src, nb, s, c->cfg.timing ? sh0.ev : nullptr, nullptr);
    }
    LST_CUDA(c, cudaGetLastError());
    sh0.ev_bin = c->cfg.timing != 0;
    for (int b = 0; b < nb; ++b) c->slots[first + b0 + b].loaded = true;
  }
  return LST_OK;
}

int lst_load_event(lst_ctx* c, int slot, const lst_hits* h, void* stream) { return lst_load_events(c, slot, 1, h, stream); }

int lst_run_stage(lst_ctx* c, int first, int n, int stage, void* stream) {
  if (!c || n < 1 || !valid_slot(c, first) || !valid_slot(c, first + n - 1) || stage < LST_MD || stage > LST_PIXEL) return LST_ERR_ARG;
  for (int s = first; s < first + n; ++s) {
    const SlotHost& h = c->slots[s];
    if (!h.loaded || h.stages_run < (stage == LST_PIXEL ? (int)LST_T5 + 1 : stage)) return LST_ERR_STATE;   // a stage needs the one before it
    if (stage == LST_PIXEL && !h.seeds_loaded) return LST_ERR_STATE;
  }
  cudaStream_t st = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  SlotHost& sh = c->slots[first];
  Params P = c->P;
  P.first_slot = first;
  if (stage == LST_PIXEL) {   // beside the linear chain: stages_run stays
    LST_CUDA(c, join_seeds(c, first, n, st));
    c->launches += launch_pixel(P, n, st, c->cfg.timing ? sh.ev + 19 : nullptr);
    LST_CUDA(c, cudaGetLastError());
    sh.ev_pix = c->cfg.timing != 0;
    for (int s = first; s < first + n; ++s) { c->slots[s].synced = false; c->slots[s].pixel_run = true; }
    return LST_OK;
  }
  if (stage == LST_CLEAN)
    c->launches += launch_clean(P, n, st, c->cfg.timing ? sh.ev + 12 : nullptr);
  else
    c->launches += launch_stage(P, n, stage, st, c->cfg.timing ? sh.ev + 4 + 2 * stage : nullptr);
  LST_CUDA(c, cudaGetLastError());
  if (c->cfg.timing) sh.ev_stage[stage] = true;
  for (int s = first; s < first + n; ++s) { c->slots[s].synced = false; c->slots[s].stages_run = stage + 1; }
  return LST_OK;
}

int lst_load_seeds(lst_ctx* c, int first, int n_ev, const lst_seeds* seeds, void* stream) {
  if (!c || n_ev < 1 || !valid_slot(c, first) || !valid_slot(c, first + n_ev - 1) || !seeds) return LST_ERR_ARG;
  for (int b = 0; b < n_ev; ++b) {
    const lst_seeds* q = seeds + b;
    if (q->n < 0) return LST_ERR_ARG;
    if (q->n > 0 && (!q->kappa || !q->cphi || !q->sphi || !q->z0 || !q->t)) return LST_ERR_ARG;
    if (!c->slots[first + b].loaded) return LST_ERR_STATE;
    if (q->n > c->cfg.cap_seeds) return LST_ERR_OVERFLOW;
  }
  cudaStream_t s = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  const Layout& L = c->P.L;
  for (int b0 = 0; b0 < n_ev; b0 += kMaxBatch) {
    const int nb = n_ev - b0 < kMaxBatch ? n_ev - b0 : kMaxBatch;
    SeedBatch src;
    std::memset(&src, 0, sizeof(src));
    for (int b = 0; b < nb; ++b) {
      const lst_seeds* q = seeds + b0 + b;
      SlotHost& sh = c->slots[first + b0 + b];
      sh.seeds_loaded = sh.pixel_run = sh.synced = false;
      sh.n_seeds_in = q->n;
      const float* in[5] = {q->kappa, q->cphi, q->sphi, q->z0, q->t};
      if (!q->on_device && q->n > 0) {
        // pinned host arrays are read by the binning kernel over PCIe (100 kB per event); pageable ones are copied first
        const void* al[5];
        bool mapped = true;
        for (int k = 0; k < 5; ++k) { al[k] = mapped_alias(in[k]); mapped = mapped && al[k]; }
        float* stage = reinterpret_cast<float*>(c->arena + (size_t)(first + b0 + b) * c->P.slot_stride + L.seed_in);
        for (int k = 0; k < 5; ++k) {
          if (mapped) { in[k] = static_cast<const float*>(al[k]); continue; }
          float* d = stage + (size_t)k * (size_t)c->cfg.cap_seeds;
          LST_CUDA(c, cudaMemcpyAsync(d, in[k], 4 * (size_t)q->n, cudaMemcpyHostToDevice, s));
          in[k] = d;
        }
      }
      src.ev[b] = SeedInput{in[0], in[1], in[2], in[3], in[4], q->n};
    }
    Params P = c->P;
    P.first_slot = first + b0;
    SlotHost& s0 = c->slots[first + b0];
    LST_CUDA(c, join_seeds(c, first + b0, nb, s));   // seeds loaded twice: the earlier binning first
    cudaStream_t side = c->seed_stream[((first + b0) / kMaxBatch) % lst_ctx::kSeedStreams];
    LST_CUDA(c, cudaEventRecord(s0.seed_fork, s));
    LST_CUDA(c, cudaStreamWaitEvent(side, s0.seed_fork, 0));
    c->launches += launch_seed_bin(P, src, nb, side, c->cfg.timing ? s0.ev + 17 : nullptr);
    LST_CUDA(c, cudaGetLastError());
    LST_CUDA(c, cudaEventRecord(s0.seed_done, side));
    s0.ev_seed = c->cfg.timing != 0;
    for (int b = 0; b < nb; ++b) {
      c->slots[first + b0 + b].seeds_loaded = true;
      c->slots[first + b0 + b].seed_owner = first + b0;
    }
  }
  return LST_OK;
}

int lst_run_batch(lst_ctx* c, int first, int n, void* stream) {
  for (int stage = LST_MD; stage <= LST_T5; ++stage) {
    const int r = lst_run_stage(c, first, n, stage, stream);
    if (r != LST_OK) return r;
  }
  return LST_OK;
}

int lst_run(lst_ctx* c, int slot, void* stream) { return lst_run_batch(c, slot, 1, stream); }

int lst_sync(lst_ctx* c, int slot, void* stream) {
  if (!valid_slot(c, slot)) return LST_ERR_ARG;
  SlotHost& sh = c->slots[slot];
  if (!sh.loaded) return LST_ERR_STATE;
  cudaStream_t s = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  LST_CUDA(c, join_seeds(c, slot, 1, s));
  const char* base = c->arena + (size_t)slot * c->P.slot_stride;
  LST_CUDA(c, cudaMemcpyAsync(sh.hdr, base + c->P.L.hdr, sizeof(SlotHeader), cudaMemcpyDeviceToHost, s));
  LST_CUDA(c, cudaStreamSynchronize(s));
  sh.synced = true;
  if (sh.hdr->overflow) return LST_ERR_OVERFLOW;
  if (sh.hdr->bad_hits) return LST_ERR_ARG;
  return LST_OK;
}

static int view_ready(lst_ctx* c, int slot, int kind) {
  if (!valid_slot(c, slot)) return LST_ERR_ARG;
  const SlotHost& sh = c->slots[slot];
  if (!sh.synced || sh.stages_run <= kind) return LST_ERR_STATE;
  if (sh.hdr->overflow) return LST_ERR_OVERFLOW;
  return LST_OK;
}

int lst_get_mds(lst_ctx* c, int slot, lst_md_view* v) {
  const int r = view_ready(c, slot, LST_MD);
  if (r != LST_OK || !v) return r != LST_OK ? r : LST_ERR_ARG;
  const Layout& L = c->P.L;
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  v->n = c->slots[slot].hdr->n[LST_MD];
  v->hits = (const int32_t*)(b + L.md_hits);
  v->module = (const int32_t*)(b + L.md_module);
  v->anchor = (const float*)(b + L.md_anchor);
  v->ur_sina = (const float*)(b + L.md_aux);
  v->dphi_dphichange = c->P.store_half ? nullptr : (const float*)(b + L.md_out);
  v->dphi_dphichange_h = c->P.store_half ? (const uint16_t*)(b + L.md_out) : nullptr;
  v->module_start = (const int32_t*)(b + L.md_start);
  return LST_OK;
}

int lst_get_segments(lst_ctx* c, int slot, lst_seg_view* v) {
  const int r = view_ready(c, slot, LST_SEG);
  if (r != LST_OK || !v) return r != LST_OK ? r : LST_ERR_ARG;
  const Layout& L = c->P.L;
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  v->n = c->slots[slot].hdr->n[LST_SEG];
  v->md = (const int32_t*)(b + L.seg_md);
  v->f = c->P.store_half ? nullptr : (const float*)(b + L.seg_f);
  v->f_h = c->P.store_half ? (const uint16_t*)(b + L.seg_f) : nullptr;
  v->md_start = (const int32_t*)(b + L.seg_start);
  return LST_OK;
}

int lst_get_triplets(lst_ctx* c, int slot, lst_t3_view* v) {
  const int r = view_ready(c, slot, LST_T3);
  if (r != LST_OK || !v) return r != LST_OK ? r : LST_ERR_ARG;
  const Layout& L = c->P.L;
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  v->n = c->slots[slot].hdr->n[LST_T3];
  v->md_kappa = (const int32_t*)(b + L.t3_pack);
  v->seg = (const int32_t*)(b + L.t3_seg);
  v->chi2rz = c->P.store_half ? nullptr : (const float*)(b + L.t3_chi2);
  v->chi2rz_h = c->P.store_half ? (const uint16_t*)(b + L.t3_chi2) : nullptr;
  v->seg_start = (const int32_t*)(b + L.t3_start);
  return LST_OK;
}

int lst_get_quintuplets(lst_ctx* c, int slot, lst_t5_view* v) {
  const int r = view_ready(c, slot, LST_T5);
  if (r != LST_OK || !v) return r != LST_OK ? r : LST_ERR_ARG;
  const Layout& L = c->P.L;
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  v->n = c->slots[slot].hdr->n[LST_T5];
  v->md = (const int32_t*)(b + L.t5_md);
  v->t3 = (const int32_t*)(b + L.t5_t3);
  v->f = c->P.store_half ? nullptr : (const float*)(b + L.t5_f);
  v->f_h = c->P.store_half ? (const uint16_t*)(b + L.t5_f) : nullptr;
  v->t3_start = (const int32_t*)(b + L.t5_start);
  return LST_OK;
}

int lst_get_track_candidates(lst_ctx* c, int slot, lst_tc_view* v) {
  const int r = view_ready(c, slot, LST_CLEAN);
  if (r != LST_OK || !v) return r != LST_OK ? r : LST_ERR_ARG;
  const Layout& L = c->P.L;
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  v->n = c->slots[slot].hdr->n_kept;
  v->t5 = (const int32_t*)(b + L.tc_list);
  v->keep = (const uint8_t*)(b + L.t5_keep);
  v->score = (const float*)(b + L.t5_score);
  return LST_OK;
}

static int pixel_ready(lst_ctx* c, int slot, int kind) {
  if (!valid_slot(c, slot) || kind < 0 || kind > 1) return LST_ERR_ARG;
  const SlotHost& sh = c->slots[slot];
  if (!sh.synced || !sh.pixel_run) return LST_ERR_STATE;
  if (sh.hdr->overflow) return LST_ERR_OVERFLOW;
  return LST_OK;
}

int lst_get_pixel_links(lst_ctx* c, int slot, int kind, lst_pix_view* v) {
  const int r = pixel_ready(c, slot, kind);
  if (r != LST_OK || !v) return r != LST_OK ? r : LST_ERR_ARG;
  const Layout& L = c->P.L;
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  v->n = c->slots[slot].hdr->n_pix[kind];
  v->link = (const int32_t*)(b + L.pix_link[kind]);
  v->f = (const float*)(b + L.pix_f[kind]);
  v->object_start = (const int32_t*)(b + L.pix_start[kind]);
  return LST_OK;
}

int lst_fetch_pixel_links(lst_ctx* c, int slot, int kind, int32_t* link_out, float* f_out, int64_t cap, void* stream) {
  const int r = pixel_ready(c, slot, kind);
  if (r != LST_OK) return r;
  const int n = c->slots[slot].hdr->n_pix[kind];
  if (n == 0) return LST_OK;
  if (cap < n) return LST_ERR_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  if (link_out) LST_CUDA(c, cudaMemcpyAsync(link_out, b + c->P.L.pix_link[kind], 8 * (size_t)n, cudaMemcpyDeviceToHost, s));
  if (f_out) LST_CUDA(c, cudaMemcpyAsync(f_out, b + c->P.L.pix_f[kind], 12 * (size_t)n, cudaMemcpyDeviceToHost, s));
  LST_CUDA(c, cudaStreamSynchronize(s));
  return LST_OK;
}

int lst_fetch_kept(lst_ctx* c, int slot, int32_t* out, int64_t cap, void* stream) {
  const int r = view_ready(c, slot, LST_CLEAN);
  if (r != LST_OK) return r;
  const int n = c->slots[slot].hdr->n_kept;
  if (n == 0) return LST_OK;
  if (!out || cap < n) return LST_ERR_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  const char* b = c->arena + (size_t)slot * c->P.slot_stride;
  LST_CUDA(c, cudaMemcpyAsync(out, b + c->P.L.tc_list, sizeof(int32_t) * (size_t)n, cudaMemcpyDeviceToHost, s));
  LST_CUDA(c, cudaStreamSynchronize(s));
  return LST_OK;
}

int lst_get_stats(lst_ctx* c, int slot, lst_stats* o) {
  if (!valid_slot(c, slot) || !o) return LST_ERR_ARG;
  SlotHost& sh = c->slots[slot];
  if (!sh.synced) return LST_ERR_STATE;
  std::memset(o, 0, sizeof(*o));
  o->n_hits = sh.hdr->n_hits;
  for (int k = 0; k < 4; ++k) { o->needed[k] = (int64_t)sh.hdr->needed[k]; o->candidates[k] = (int64_t)sh.hdr->cand[k]; o->evaluated[k] = (int64_t)sh.hdr->eval[k]; o->rewalks[k] = (int64_t)sh.hdr->rewalk[k]; }
  o->overflow = sh.hdr->overflow;
  o->bad_hits = sh.hdr->bad_hits;
  o->n_kept = sh.stages_run > LST_CLEAN ? sh.hdr->n_kept : 0;
  if (sh.seeds_loaded) o->n_seeds = sh.hdr->n_seeds;
  if (sh.pixel_run)
    for (int k = 0; k < 2; ++k) {
      o->pix_needed[k] = (int64_t)sh.hdr->needed_pix[k]; o->pix_candidates[k] = (int64_t)sh.hdr->cand_pix[k];
      o->pix_evaluated[k] = (int64_t)sh.hdr->eval_pix[k]; o->pix_rewalks[k] = (int64_t)sh.hdr->rewalk_pix[k];
    }
  if (c->cfg.timing) {
    if (sh.ev_bin) {
      cudaEventElapsedTime(&o->stage_ms[0], sh.ev[0], sh.ev[3]);
      for (int k = 0; k < 3; ++k) cudaEventElapsedTime(&o->kernel_ms[k], sh.ev[k], sh.ev[k + 1]);
    }
    if (sh.ev_stage[4])
      for (int k = 0; k < 4; ++k) cudaEventElapsedTime(&o->kernel_ms[7 + k], sh.ev[12 + k], sh.ev[13 + k]);
    if (sh.ev_seed) cudaEventElapsedTime(&o->pix_ms[0], sh.ev[17], sh.ev[18]);
    if (sh.ev_pix) { cudaEventElapsedTime(&o->pix_ms[1], sh.ev[19], sh.ev[20]); cudaEventElapsedTime(&o->pix_ms[2], sh.ev[20], sh.ev[21]); }
    for (int st = 0; st < 4; ++st)
      if (sh.ev_stage[st]) {
        cudaEvent_t* e = sh.ev + 4 + 2 * st;
        cudaEventElapsedTime(&o->stage_ms[1 + st], e[0], e[1]);
        o->kernel_ms[3 + st] = o->stage_ms[1 + st];
      }
    cudaGetLastError();
  }
  return LST_OK;
}

static const int kHitsPerObject[5] = {2, 4, 6, 10, 10};     // [4]: the kept quintuplets (LST_CLEAN)
static const int kValuesPerObject[5] = {4, 4, 2, 5, 5};

int lst_sync_batch(lst_ctx* c, int first, int n, void* stream) {
  if (!c || n < 1 || !valid_slot(c, first) || !valid_slot(c, first + n - 1)) return LST_ERR_ARG;
  for (int s = first; s < first + n; ++s)
    if (!c->slots[s].loaded) return LST_ERR_STATE;
  cudaStream_t st = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  LST_CUDA(c, join_seeds(c, first, n, st));
  // the n headers in ONE strided copy: they sit slot_stride apart on the device, contiguous in the pinned mirror
  LST_CUDA(c, cudaMemcpy2DAsync(c->pinned + first, sizeof(SlotHeader), c->arena + (size_t)first * c->P.slot_stride + c->P.L.hdr,
                                c->P.slot_stride, sizeof(SlotHeader), (size_t)n, cudaMemcpyDeviceToHost, st));
  LST_CUDA(c, cudaStreamSynchronize(st));
  int status = LST_OK;
  for (int s = first; s < first + n; ++s) {
    SlotHost& sh = c->slots[s];
    sh.synced = true;
    if (status == LST_OK && sh.hdr->overflow) status = LST_ERR_OVERFLOW;
  }
  if (status == LST_OK)
    for (int s = first; s < first + n; ++s)
      if (c->slots[s].hdr->bad_hits) { status = LST_ERR_ARG; break; }
  return status;
}

static inline int count_of(const SlotHeader* h, int kind) { return kind == LST_CLEAN ? h->n_kept : h->n[kind]; }

int lst_fetch_batch(lst_ctx* c, int first, int n, int kind, int32_t* const* idx_out, void* const* val_out,
                    const int64_t* cap_objects, int32_t* counts, int wait, void* stream) {
  if (!c || n < 1 || !valid_slot(c, first) || !valid_slot(c, first + n - 1) || kind < LST_MD || kind > LST_CLEAN || !cap_objects)
    return LST_ERR_ARG;
  for (int s = first; s < first + n; ++s)
    if (!c->slots[s].loaded || c->slots[s].stages_run <= kind) return LST_ERR_STATE;
  bool all_synced = true;
  for (int s = first; s < first + n; ++s) all_synced = all_synced && c->slots[s].synced;
  if (!all_synced) {
    const int r = lst_sync_batch(c, first, n, stream);
    if (r == LST_ERR_CUDA || r == LST_ERR_STATE) return r;
  }
  int n_max = 0;
  for (int b = 0; b < n; ++b) {
    const SlotHeader* h = c->slots[first + b].hdr;
    if (h->overflow) return LST_ERR_OVERFLOW;
    const int nk = count_of(h, kind);
    if (counts) counts[b] = nk;
    if (nk > cap_objects[b] && ((idx_out && idx_out[b]) || (val_out && val_out[b]))) return LST_ERR_ARG;
    n_max = nk > n_max ? nk : n_max;
  }
  cudaStream_t st = (cudaStream_t)stream;
  LST_CUDA(c, cudaSetDevice(c->device));
  const Layout& L = c->P.L;
  Params P = c->P;
  P.first_slot = first;
  // Pinned (mapped) host buffers are written by ONE kernel per 16 slots (k_fetch_direct); what is left (pageable
  // buffers) goes through the slot's scratch area and the copy engine, below.
  std::vector<int32_t*> idx_dma(idx_out ? idx_out : nullptr, idx_out ? idx_out + n : nullptr);
  std::vector<void*> val_dma(val_out ? val_out : nullptr, val_out ? val_out + n : nullptr);
  for (int b0 = 0; b0 < n && n_max > 0; b0 += kMaxBatch) {
    const int nb = n - b0 < kMaxBatch ? n - b0 : kMaxBatch;
    OutTable T;
    std::memset(&T, 0, sizeof(T));
    bool any = false;
    for (int b = 0; b < nb; ++b) {
      if (count_of(c->slots[first + b0 + b].hdr, kind) == 0) continue;
      if (idx_out && idx_out[b0 + b])
        if (void* a = const_cast<void*>(mapped_alias(idx_out[b0 + b]))) { T.idx[b] = static_cast<int*>(a); idx_dma[b0 + b] = nullptr; any = true; }
      if (val_out && val_out[b0 + b])
        if (void* a = const_cast<void*>(mapped_alias(val_out[b0 + b]))) { T.val[b] = a; val_dma[b0 + b] = nullptr; any = true; }
    }
    if (!any) continue;
    Params Pd = c->P;
    Pd.first_slot = first + b0;
    c->launches += launch_fetch_direct(Pd, T, kind, nb, st);
    LST_CUDA(c, cudaGetLastError());
  }
  bool idx_left = false, val_left = false;
  for (int b = 0; b < n; ++b) {
    const bool has = count_of(c->slots[first + b].hdr, kind) > 0;
    idx_left = idx_left || (has && idx_out && idx_dma[b]);
    val_left = val_left || (has && val_out && val_dma[b]);
  }
  idx_out = idx_left ? idx_dma.data() : nullptr;
  val_out = val_left ? val_dma.data() : nullptr;
  // The slot's scratch area holds one gathered table at a time: stream order keeps the second gather behind the
  // first copy.
  if (idx_out && n_max > 0) {
    c->launches += launch_gather_hits(P, kind, n_max, n, st);
    LST_CUDA(c, cudaGetLastError());
    for (int b = 0; b < n; ++b) {
      const int nk = count_of(c->slots[first + b].hdr, kind);
      if (!idx_out[b] || nk == 0) continue;
      const char* base = c->arena + (size_t)(first + b) * c->P.slot_stride;
      LST_CUDA(c, cudaMemcpyAsync(idx_out[b], base + L.scratch, sizeof(int32_t) * (size_t)nk * kHitsPerObject[kind], cudaMemcpyDeviceToHost, st));
    }
  }
  if (val_out && n_max > 0) {
    // LS and T5 payloads are stored in the output layout (in either precision): copied straight from the store
    const bool packed = kind == LST_MD || kind == LST_T3 || kind == LST_CLEAN;
    if (packed) {
      c->launches += launch_pack_values(P, kind, n_max, n, st);
      LST_CUDA(c, cudaGetLastError());
    }
    const size_t src_off = packed ? L.scratch : (kind == LST_SEG ? L.seg_f : L.t5_f);
    const size_t elem = c->P.store_half ? 2 : 4;
    for (int b = 0; b < n; ++b) {
      const int nk = count_of(c->slots[first + b].hdr, kind);
      if (!val_out[b] || nk == 0) continue;
      const char* base = c->arena + (size_t)(first + b) * c->P.slot_stride;
      LST_CUDA(c, cudaMemcpyAsync(val_out[b], base + src_off, elem * (size_t)nk * kValuesPerObject[kind], cudaMemcpyDeviceToHost, st));
    }
  }
  if (wait) LST_CUDA(c, cudaStreamSynchronize(st));
  return LST_OK;
}

int lst_fetch_hit_indices(lst_ctx* c, int slot, int kind, int32_t* out, int64_t cap, void* stream) {
  if (kind < LST_MD || kind > LST_T5) return LST_ERR_ARG;
  const int r = view_ready(c, slot, kind);
  if (r != LST_OK) return r;
  const int n = c->slots[slot].hdr->n[kind];
  if (n == 0) return LST_OK;
  if (!out || cap < n) return LST_ERR_ARG;
  int32_t* outs[1] = {out};
  const int64_t caps[1] = {cap};
  return lst_fetch_batch(c, slot, 1, kind, outs, nullptr, caps, nullptr, 1, stream);
}

int lst_fetch_values(lst_ctx* c, int slot, int kind, void* out, int64_t cap, void* stream) {
  if (kind < LST_MD || kind > LST_T5) return LST_ERR_ARG;
  const int r = view_ready(c, slot, kind);
  if (r != LST_OK) return r;
  const int n = c->slots[slot].hdr->n[kind];
  if (n == 0) return LST_OK;
  if (!out || cap < n) return LST_ERR_ARG;
  void* outs[1] = {out};
  const int64_t caps[1] = {cap};
  return lst_fetch_batch(c, slot, 1, kind, nullptr, outs, caps, nullptr, 1, stream);
}

int lst_grown_config(lst_ctx* c, int slot, lst_config* out) {
  if (!valid_slot(c, slot) || !out) return LST_ERR_ARG;
  const SlotHost& sh = c->slots[slot];
  if (!sh.synced) return LST_ERR_STATE;
  *out = c->cfg;
  auto grow = [](int32_t& cap, unsigned long long needed) {
    if (needed <= (unsigned long long)cap) return;
    unsigned long long want = (needed + needed / 4 + 1023) / 1024 * 1024;
    if (want > (unsigned long long)kMaxCap) want = (unsigned long long)kMaxCap;
    cap = (int32_t)want;
  };
  grow(out->cap_md, sh.hdr->needed[LST_MD]);
  grow(out->cap_seg, sh.hdr->needed[LST_SEG]);
  grow(out->cap_t3, sh.hdr->needed[LST_T3]);
  grow(out->cap_t5, sh.hdr->needed[LST_T5]);
  if (sh.pixel_run) {
    grow(out->cap_pt3, sh.hdr->needed_pix[0]);
    grow(out->cap_pt5, sh.hdr->needed_pix[1]);
  }
  return LST_OK;
}

int lst_arena_bytes(lst_ctx* c, int64_t* total, int64_t* per_slot) {
  if (!c) return LST_ERR_ARG;
  if (total) *total = (int64_t)c->arena_bytes;
  if (per_slot) *per_slot = (int64_t)c->P.slot_stride;
  return LST_OK;
}

int64_t lst_launch_count(lst_ctx* c) { return c ? (int64_t)c->launches.load() : 0; }
int lst_last_cuda_error(lst_ctx* c) { return c ? c->last_cuda.load() : 0; }

const char* lst_strerror(int s) {
  switch (s) {
    case LST_OK: return "ok";
    case LST_ERR_ARG: return "invalid argument or input (geometry, module map, slot, module id, side)";
    case LST_ERR_CUDA: return "CUDA runtime error (see lst_last_cuda_error)";
    case LST_ERR_OVERFLOW: return "a per-slot capacity was exceeded; outputs of the slot are invalid";
    case LST_ERR_STATE: return "call out of order (load -> run -> sync -> get)";
    case LST_ERR_NOMEM: return "arena allocation failed";
    case LST_ERR_LIMIT: return "size beyond the fixed maximum of the entry point that allocates nothing (LST_MAP_STATIC_MAX_MODULES)";
  }
  return "unknown status";
}

const char* lst_version(void) { return "lst-b200 0.1 (sm_100a)"; }

}  // extern "C"
