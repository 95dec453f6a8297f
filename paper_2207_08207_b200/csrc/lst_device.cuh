// lst_device.cuh -- device-side data layout of one event slot and the kernel launch parameters.
//
// One arena (allocated once in lst_create) holds n_slots identical slots;
// every array of a slot sits at a fixed byte offset from the slot base (struct Layout), so a
// kernel finds slot s at arena + s * slot_stride and needs no per-slot pointer table.  The
// batch index (which slot of a batch) is blockIdx.y of every kernel.
//
// Hit store (per slot): hits are binned by (side, module) -- all lower-sensor hits first, in
// module order, then all upper-sensor hits -- and ordered inside a bin by their azimuth
// relative to the module normal (`key`), ties by original index.  Lower hit i of the event is
// simply element i: the MD kernel's owners are the lower hits.
//   hit4[i]      = (x, y, z, r)            float4
//   hit_key[i]   = azimuth - module azimuth float   (FLT_MAX for non-finite x / y)
//   hit_orig[i]  = original index           int
//   hit_module[i]                           int
// Object store, "SoA of small vectors": each class keeps one array per GROUP of fields that
// are always read together, packed to 8 or 16 bytes so one vector load fetches the group
// (PAPER.md:139-141 argues for SoA on V100; on sm_100a the unit that matters is the 16-B
// vector / 32-B sector):
// Fields marked [h] are pure outputs (no later selection reads them): with Params::store_half they are stored as IEEE
// binary16 (round to nearest even of the fp32 value) in the first half of the same array (DESIGN.md section 1 [H]).
//   MD     md_anchor  = (x, y, z, r) of anchor  float4   ordered by (module, key of anchor hit)
//          md_aux     = (r_upper, sinA)         float2
//          md_key     = key of the anchor hit   float    (the segment search window runs on it)
//          md_hits    = (orig lower, orig upper)int2
//          md_out     = (dphi, dphichange)      float2   [h]
//          md_module                            int
//   LS     seg_md     = (inner MD, outer MD)    int2
//          seg_f      = (sinS, z0, dphi, dphichange) float4   [h]
//   T3     t3_pack    = (MD1, MD2, MD3, kappa)  int4 (kappa as bits)
//          t3_seg     = (seg a, seg b)          int2
//          t3_chi2                              float    [h]
//   T5     t5_md[5], t5_t3 = (A, B) int2, t5_f[5] = kA, kB, kfit, chi2xy, chi2rz [h], t5_score = chi2xy + chi2rz (fp32, read by [D])
// CSR offsets: bin_start[2*n_modules+1], md_start[n_modules+1], seg_start[cap_md+1] (by inner
// MD), t3_start[cap_seg+1] (by first segment), t5_start[cap_t3+1] (by inner triplet).
// mod_info[m] = (first MD, end MD, smallest key, largest key of the module's lower hits).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "lst_cuts.cuh"

namespace lst {

constexpr int kChunk = 32;        // owners (lower hits / MDs / segments / triplets) per warp chunk
constexpr int kMaxBatch = 16;     // events per launch of the a0 kernels (pointer table in the launch parameters)
constexpr int kMaxRow = 64;       // longest module-map row accepted
constexpr int kMaxCap = 1 << 26;  // largest per-slot capacity: object indices are packed into 26 bits
enum { LST_MD_ = 0, LST_SEG_ = 1, LST_T3_ = 2, LST_T5_ = 3, LST_CLEAN_ = 4, LST_PIXEL_ = 5 };  // == LST_MD .. LST_PIXEL of lst.h
// [P] pixel line segments (seeds) are binned by (curvature band, azimuth of their direction at the beam line): kSeedBands bands
// x kSeedPhiBins uniform azimuth bins over (-pi, pi], a seed filed under every band an object within pix_dkappa_max of it can
// sit in; then bin kSeedBins = seeds whose (cos, sin) is not a unit vector (no azimuth window can be derived for them: every
// object looks at them), then bin kSeedBins + 1 = seeds that no object can accept (non-finite or zero direction, NaN curvature).
constexpr int kSeedPhiBins = 512, kSeedBands = 16, kSeedBins = kSeedPhiBins * kSeedBands;

struct SlotHeader {
  int n_hits;                     // valid hits binned
  int n_lower;                    // of which on the lower sensor (= bin_start[n_modules])
  int n[4];                       // objects stored (clamped to capacity): MD, LS, T3, T5
  int overflow;                   // bit k: class k exceeded its capacity
  int bad_hits;                   // hits dropped (module id / side out of range)
  unsigned long long needed[4];   // objects that passed (unclamped)
  unsigned long long cand[4];     // candidates of the search space (map-restricted pairs)
  unsigned long long eval[4];     // candidates the selection was evaluated on (after windowing)
  unsigned long long rewalk[4];   // chunks whose objects did not fit the shared-memory stash (walked twice)
  // per side, per layer: range of r over the finite hits, as float bit patterns;
  // r_min is stored as 0x7f800000 - bits so that the zeroed header means "+inf"
  int r_min_inv[2][6];
  int r_max[2][6];
  int key_absmax[6];              // per layer: largest |key| of the finite lower-sensor hits, as float bits (directly after r_max: one flush loop)
  unsigned int done[8];           // "last block done" tickets, self-resetting (never zeroed with the header)
  unsigned int ticket[4];         // next chunk of the single-pass kernels (zeroed with the header)
  int n_kept;                     // quintuplets kept by the duplicate cleaning (stage LST_CLEAN)
  unsigned int bad_acc;           // invalid hits seen by k_bin_count so far; moved to bad_hits and cleared by its last block
  // [P] pixel links, index 0 = pixel triplets (seed + T3), 1 = pixel quintuplets (seed + T5); written by k_seed_bin / k_pix
  int n_seeds;                    // seeds loaded (lst_load_seeds)
  int n_pix[2];                   // links stored (clamped to capacity); overflow bits 4, 5
  unsigned int ticket_pix[2];
  unsigned long long needed_pix[2], cand_pix[2], eval_pix[2], rewalk_pix[2];
};

struct Layout {
  int n_modules, n_bins;
  int cap_hits, cap_md, cap_seg, cap_t3, cap_t5;
  int cap_seeds, cap_pix[2];      // [P] seeds per slot; pixel triplets / pixel quintuplets per slot
  int n_chunk[4];                 // ceil(cap of the OWNER class / kChunk): hits, MD, LS, T3
  int n_chunk_pix[2];             // owners of the pixel stage: T3, T5
  // byte offsets from the slot base (all multiples of 256)
  size_t hdr, bin_cnt, bin_start, lb[4];      // header; bin counters (self-cleaning); bin offsets; look-back words (contiguous)
  size_t lb_bytes;                            // bytes of the four look-back arrays, zeroed by k_bin_scatter
  size_t in_x, in_y, in_z, in_module, in_side;// destination of host -> device copies of the caller's arrays (copy-engine paths)
  size_t rec4, recb, reck;                    // per input hit: (x, y, z, key), (bin, arrival rank in the bin), key again (dense)
  size_t tmp_ki, tmp_bin;                     // per hit at its unsorted place in the bin: (original index, sortable key), bin
  size_t hit4, hit_key, hit_orig, hit_module;
  size_t md_start, mod_info, md_anchor, md_aux, md_key, md_hits, md_out, md_module;
  size_t seg_start, seg_md, seg_f;
  size_t t3_start, t3_pack, t3_seg, t3_chi2;
  size_t t5_start, t5_md, t5_t3, t5_f;
  size_t t5_kfit;                             // fitted curvature in fp32 whatever the store ([P] P1 reads it)
  size_t t5_hits, t5_score, t5_keep, tc_list, inc_start, inc_cur, inc_list;   // duplicate cleaning
  // [P]: copy destination of host seed arrays (5 x cap_seeds floats); seeds ordered by azimuth bin: (kappa, cos, sin, z0),
  // (t, original index); bin offsets [kSeedBins + 3]; look-back words of the two link kernels (contiguous, cleared by
  // k_seed_bin); per kind: CSR offsets by outer object, links (seed, object), values (chi2xy, chi2rz, kappa_obj - kappa)
  size_t seed_in, seed_rec4, seed_rec2, seed_bin_start, lb_pix[2], lb_pix_bytes;
  size_t pix_start[2], pix_link[2], pix_f[2];
  size_t scratch;
  size_t slot_bytes;
};

// Launch parameters, passed by value (constant bank): no per-launch device reads to find data.
struct Params {
  char* arena;
  size_t slot_stride;
  Layout L;
  Cuts cuts;
  const signed char* mod_layer;  // [n_modules]
  const float2* mod_cs;          // [n_modules] (cos, sin) of the azimuth of the module normal
  const int* map_offsets;        // [n_modules + 1] module map, CSR
  const int* map_targets;        // [map_offsets[n_modules]] rows ordered by (map_dphi, target): the entries an inner MD can reach are one run
  const float* map_dphi;         // [map_offsets[n_modules]] azimuth(source normal) - azimuth(target normal), in (-pi, pi], ascending per row
  const int* map_targets_asc;    // the same rows ordered by target (k_seg's direct walk: segments arrive in CSR order)
  const float* map_dphi_asc;     // azimuth offsets in that order
  int first_slot;
  int dup_min_shared;            // [D] D4: quintuplets sharing at least this many original hits are duplicates
  int store_half;                // [H] output floats that no selection reads are stored as binary16
  int four_launches;             // lst_config.launches_in_flight >= 4: stage grids sized for four launches side by side (host side only)
  int live_modules[3];           // modules 0 .. live_modules[k]-1 are exactly those on layers <= 1 (k = 0) / <= 3 (k = 1) / <= 4 (k = 2) when the
                                 // module ids are ordered by layer, else n_modules: owners of the quintuplet and pixel / triplet / segment
                                 // kernel behind the corresponding CSR prefix have no candidates
};

// Typed access to one slot.
struct Slot {
  char* b;
  const Layout& L;
  __device__ __forceinline__ Slot(const Params& P, int batch_index)
      : b(P.arena + (size_t)(P.first_slot + batch_index) * P.slot_stride), L(P.L) {}
  template <class T>
  __device__ __forceinline__ T* at(size_t off) const { return reinterpret_cast<T*>(b + off); }
  __device__ __forceinline__ SlotHeader* hdr() const { return at<SlotHeader>(L.hdr); }
  __device__ __forceinline__ unsigned* bin_cnt() const { return at<unsigned>(L.bin_cnt); }
  __device__ __forceinline__ unsigned* bin_start() const { return at<unsigned>(L.bin_start); }
  __device__ __forceinline__ unsigned long long* lb(int kind) const { return at<unsigned long long>(L.lb[kind]); }
  __device__ __forceinline__ float4* rec4() const { return at<float4>(L.rec4); }
  __device__ __forceinline__ int2* recb() const { return at<int2>(L.recb); }
  __device__ __forceinline__ float* reck() const { return at<float>(L.reck); }
  __device__ __forceinline__ int2* tmp_ki() const { return at<int2>(L.tmp_ki); }
  __device__ __forceinline__ int* tmp_bin() const { return at<int>(L.tmp_bin); }
  __device__ __forceinline__ float4* hit4() const { return at<float4>(L.hit4); }
  __device__ __forceinline__ float* hit_key() const { return at<float>(L.hit_key); }
  __device__ __forceinline__ int* hit_orig() const { return at<int>(L.hit_orig); }
  __device__ __forceinline__ int* hit_module() const { return at<int>(L.hit_module); }
  __device__ __forceinline__ int* md_start() const { return at<int>(L.md_start); }
  __device__ __forceinline__ int4* mod_info() const { return at<int4>(L.mod_info); }
  __device__ __forceinline__ float4* md_anchor() const { return at<float4>(L.md_anchor); }
  __device__ __forceinline__ float2* md_aux() const { return at<float2>(L.md_aux); }
  __device__ __forceinline__ float* md_key() const { return at<float>(L.md_key); }
  __device__ __forceinline__ int2* md_hits() const { return at<int2>(L.md_hits); }
  __device__ __forceinline__ float2* md_out() const { return at<float2>(L.md_out); }
  __device__ __forceinline__ int* md_module() const { return at<int>(L.md_module); }
  __device__ __forceinline__ int* seg_start() const { return at<int>(L.seg_start); }
  __device__ __forceinline__ int2* seg_md() const { return at<int2>(L.seg_md); }
  __device__ __forceinline__ float4* seg_f() const { return at<float4>(L.seg_f); }
  __device__ __forceinline__ int* t3_start() const { return at<int>(L.t3_start); }
  __device__ __forceinline__ int4* t3_pack() const { return at<int4>(L.t3_pack); }
  __device__ __forceinline__ int2* t3_seg() const { return at<int2>(L.t3_seg); }
  __device__ __forceinline__ float* t3_chi2() const { return at<float>(L.t3_chi2); }
  __device__ __forceinline__ int* t5_start() const { return at<int>(L.t5_start); }
  __device__ __forceinline__ int* t5_md() const { return at<int>(L.t5_md); }
  __device__ __forceinline__ int2* t5_t3() const { return at<int2>(L.t5_t3); }
  __device__ __forceinline__ float* t5_f() const { return at<float>(L.t5_f); }
  __device__ __forceinline__ int* t5_hits() const { return at<int>(L.t5_hits); }
  __device__ __forceinline__ float* t5_score() const { return at<float>(L.t5_score); }
  __device__ __forceinline__ float* t5_kfit() const { return at<float>(L.t5_kfit); }
  __device__ __forceinline__ unsigned char* t5_keep() const { return at<unsigned char>(L.t5_keep); }
  __device__ __forceinline__ int* tc_list() const { return at<int>(L.tc_list); }
  __device__ __forceinline__ int* inc_start() const { return at<int>(L.inc_start); }
  __device__ __forceinline__ int* inc_cur() const { return at<int>(L.inc_cur); }
  __device__ __forceinline__ int2* inc_list() const { return at<int2>(L.inc_list); }
  __device__ __forceinline__ int* scratch() const { return at<int>(L.scratch); }
  __device__ __forceinline__ float4* seed_rec4() const { return at<float4>(L.seed_rec4); }
  __device__ __forceinline__ float2* seed_rec2() const { return at<float2>(L.seed_rec2); }
  __device__ __forceinline__ int* seed_bin_start() const { return at<int>(L.seed_bin_start); }
  __device__ __forceinline__ unsigned long long* lb_pix(int kind) const { return at<unsigned long long>(L.lb_pix[kind]); }
  __device__ __forceinline__ int* pix_start(int kind) const { return at<int>(L.pix_start[kind]); }
  __device__ __forceinline__ int2* pix_link(int kind) const { return at<int2>(L.pix_link[kind]); }
  __device__ __forceinline__ float* pix_f(int kind) const { return at<float>(L.pix_f[kind]); }
};

// Raw input arrays of one event (caller's device pointers, mapped host memory, or the slot's copy destination).
struct HitInput {
  const float* x;
  const float* y;
  const float* z;
  const int* module;
  const unsigned char* side;
  int n;
  int stage;   // != 0: the arrays are mapped (pinned) host memory, read by k_bin_count over PCIe
};
// Inputs of a batch of events: slot first_slot + b reads ev[b].
struct HitBatch {
  HitInput ev[kMaxBatch];
};

// Seed arrays of one event (caller's device pointers, mapped host memory, or the slot's copy destination).
struct SeedInput {
  const float* kappa;
  const float* cphi;
  const float* sphi;
  const float* z0;
  const float* t;
  int n;
};
struct SeedBatch {
  SeedInput ev[kMaxBatch];
};

// Host-callable launchers (lst_kernels.cu). Each returns the number of kernels it launched.
// `ev` (optional, timing mode): ev[0] is recorded before the first kernel, ev[k + 1] after kernel k.
// `src`: the arrays k_bin_count reads (device, or mapped host memory with stage = 1); it is the only kernel that touches
// them.  `stage` (non-null when k_bin_count reads host memory): the library's stage-in stream and the two events that fork it
// from / join it to `s`.
struct StageIn {
  cudaStream_t stream;
  cudaEvent_t before, after;
};
int launch_bin(const Params& P, const HitBatch& src, int n_batch, cudaStream_t s, cudaEvent_t* ev,
               const StageIn* stage);   // 3 kernels
int launch_stage(const Params& P, int n_batch, int stage, cudaStream_t s, cudaEvent_t* ev);          // 1 kernel
// Duplicate cleaning [D]: 6 kernels (prepare, count, scan, fill, mark, list); ev[0..4] around the four steps.
int launch_clean(const Params& P, int n_batch, cudaStream_t s, cudaEvent_t* ev);
// [P]: seeds of a batch to azimuth bins (1 kernel; ev[0..1]); pixel triplets + pixel quintuplets (2 kernels; ev[0..2]).
int launch_seed_bin(const Params& P, const SeedBatch& src, int n_batch, cudaStream_t s, cudaEvent_t* ev);
int launch_pixel(const Params& P, int n_batch, cudaStream_t s, cudaEvent_t* ev);
// Per slot of a batch: device-visible aliases of pinned host buffers for the hit-index tuples / the float payload
// (null = that table is not wanted there, or goes through the scratch area and the copy engine).
struct OutTable {
  int* idx[kMaxBatch];
  void* val[kMaxBatch];          // fp32 values, or binary16 when Params::store_half
};
int launch_fetch_direct(const Params& P, const OutTable& T, int kind, int n_batch, cudaStream_t s);
int launch_gather_hits(const Params& P, int kind, int n_max, int n_batch, cudaStream_t s);   // slots first_slot .. + n_batch - 1
int launch_pack_values(const Params& P, int kind, int n_max, int n_batch, cudaStream_t s);

}  // namespace lst
