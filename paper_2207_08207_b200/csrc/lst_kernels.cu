// lst_kernels.cu -- sm_100a kernels of the LST hot path (DESIGN.md sections 5-7).
//
// Hits and mini-doublets are kept ordered by azimuth inside their module, so the MD and the
// segment stage look only at a window of candidates found by binary search (DESIGN.md
// section 6); every candidate in a window goes through the exact SPEC selection.
//
// Every stage is ONE single-pass kernel built from the same warp-level pipeline
// (DESIGN.md section 7):
//   * a warp takes a chunk of 32 consecutive OWNERS (lower hits / inner MDs / first segments /
//     inner triplets) from a ticket counter; each owner has a contiguous range of candidates;
//   * the ranges are flattened: a warp scan numbers the candidates, and every tile of 32
//     candidates finds its owners with one redux + popc (no search, no barrier), so all 32 lanes
//     evaluate one candidate each whatever the occupancy skew between owners;
//     (the segment kernel's first level is the exception: lane = owner, the warp steps through the
//     owners' map rows in lockstep);
//   * where a cheap test removes most candidates (module key ranges and windows for segments, the
//     curvature match for quintuplets) survivors are compacted into a small shared-memory
//     queue and the expensive selection runs on full tiles of survivors;
//   * what passes is kept, in (owner, candidate) order, in a shared-memory stash until a
//     decoupled look-back over the chunk totals has told the warp where its objects start;
//     objects are then written once, contiguous per owner (CSR), in a deterministic order.  The
//     emit is DEFERRED by one chunk: the total is published right after the walk, the warp walks
//     its next chunk, and only then resolves the base of the previous one (second stash), so the
//     ordered-output wait has a whole walk of slack (two walks of slack, or an extra non-blocking
//     attempt right after the walk, measured slower: the inclusive prefixes come later / cost a
//     round trip);
// No global atomic is issued per candidate or per object, and no block-wide barrier is used:
// warps are independent, compaction is ballot + popc.
//
// blockIdx.y = index of the event within the batch (lst_run_batch): all events of a batch go
// through one launch per kernel.
#include <cuda_fp16.h>

#include <cstddef>

#include "lst_device.cuh"

namespace lst {

constexpr unsigned kFull = 0xffffffffu;

// ------------------------------------------------------------------------------------------
// small device utilities
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned lane_id() { return threadIdx.x & 31u; }
__device__ __forceinline__ unsigned lanemask_lt() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}
__device__ __forceinline__ unsigned lanemask_le() {
  unsigned m;
  asm("mov.u32 %0, %%lanemask_le;" : "=r"(m));
  return m;
}

// Order-preserving map of a float's bit pattern to an unsigned integer (and back): (key, original index) then
// compares as ONE 64-bit integer in the ranking loop of k_bin_order.  Keys are finite or the 3e38 sentinel; -0 sorts
// just before +0, which only permutes hits whose azimuths are equal.
__device__ __forceinline__ unsigned sortable_of(float f) {
  const unsigned b = __float_as_uint(f);
  return b ^ ((unsigned)((int)b >> 31) | 0x80000000u);
}
__device__ __forceinline__ float float_of_sortable(unsigned u) {
  return __uint_as_float(u ^ ((u & 0x80000000u) ? 0x80000000u : 0xffffffffu));
}

__device__ __forceinline__ int warp_incl_scan(int v) {
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    int t = __shfl_up_sync(kFull, v, d);
    if ((int)lane_id() >= d) v += t;
  }
  return v;
}
__device__ __forceinline__ int warp_excl_scan(int v, int& total) {
  const int incl = warp_incl_scan(v);
  total = __shfl_sync(kFull, incl, 31);
  return incl - v;
}
__device__ __forceinline__ unsigned long long warp_sum_ull(unsigned long long v) {
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) v += __shfl_down_sync(kFull, v, d);
  return v;
}

// In-place exclusive scan of the ints a[0 .. n] (a[n] must be 0 on entry and receives the total)
// by the whole block.  The array is padded with zeros to a multiple of 4 ints (the slot layout rounds
// every array up to 256 bytes).  The values were written by other blocks: ld.cg.  Returns the total.
// One block runs this while the rest of the event's grid has retired, so what counts is its latency: a
// tile of NT x kPer int4 is loaded with all loads in flight at once (kPer independent 16-byte loads per
// thread, blocked layout; 1024 x 3 covers the 12 241 bin counters of the BASELINE geometry in one tile), scanned in registers + one block scan, and written back.
template <int NT, int kPer>
__device__ int block_scan_array4(int* a, int n) {
  constexpr int W = NT / 32;
  __shared__ int warp_tot[W];
  __shared__ int s_carry;
  int4* a4 = reinterpret_cast<int4*>(a);
  const int n4 = (n + 1 + 3) / 4;
  const int w = threadIdx.x >> 5, lane = (int)lane_id();
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int t0 = 0; t0 < n4; t0 += NT * kPer) {
    const int j0 = t0 + (int)threadIdx.x * kPer;
    int4 v[kPer];
#pragma unroll
    for (int k = 0; k < kPer; ++k) v[k] = (j0 + k < n4) ? __ldcg(a4 + j0 + k) : make_int4(0, 0, 0, 0);
    int mine = 0;
#pragma unroll
    for (int k = 0; k < kPer; ++k) mine += (v[k].x + v[k].y) + (v[k].z + v[k].w);
    const int incl = warp_incl_scan(mine);
    if (lane == 31) warp_tot[w] = incl;
    __syncthreads();
    int ex = s_carry + incl - mine, tile_total = 0;
#pragma unroll 8
    for (int i = 0; i < W; ++i) {
      const int t = warp_tot[i];
      ex += (i < w) ? t : 0;
      tile_total += t;
    }
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
      if (j0 + k < n4) a4[j0 + k] = make_int4(ex, ex + v[k].x, ex + v[k].x + v[k].y, ex + v[k].x + v[k].y + v[k].z);
      ex += (v[k].x + v[k].y) + (v[k].z + v[k].w);
    }
    __syncthreads();
    if (threadIdx.x == 0) s_carry += tile_total;
    __syncthreads();
  }
  return s_carry;
}

// Ticket: true in every thread of the block that finishes last among `n_blocks`.
__device__ __forceinline__ bool last_block_done(unsigned* counter, unsigned n_blocks) {
  __shared__ bool is_last;
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();   // release: cumulative over what the block's threads wrote before the barrier (as in a grid-wide sync)
    const unsigned t = atomicAdd(counter, 1u);
    is_last = (t == n_blocks - 1);
    if (is_last) atomicExch(counter, 0u);
  }
  __syncthreads();
  const bool r = is_last;
  if (r) __threadfence();
  return r;
}

__device__ __forceinline__ void publish_total(SlotHeader* h, int kind, int total, int cap) {
  h->needed[kind] = (unsigned long long)total;
  h->n[kind] = min(total, cap);
  if (total > cap) atomicOr(&h->overflow, 1 << kind);
}

// ------------------------------------------------------------------------------------------
// search windows.  A window is a conservative superset of what the SPEC
// selection can accept, derived from the selection's own inequalities and the per-event range
// of r per (side, layer); every candidate inside it goes through the exact SPEC selection, so
// the object set does not depend on the window.  Geometry of a pair seen from the beam line:
// with alpha the angle between the inner position vector and the inner->outer displacement
// (sin alpha is the cut variable sinA / sinS) and delta the azimuth difference,
//     delta = alpha - asin((r_in / r_out) sin alpha)          (law of sines; dot > 0, r_out > r_in)
// which grows with alpha, and for alpha > 0 with r_out.
// ------------------------------------------------------------------------------------------
__device__ __forceinline__ float delta_of(float s, float ratio) {
  return asinf(s) - asinf(ratio * s);
}

__device__ __forceinline__ int lower_bound_f(const float* a, int lo, int hi, float v) {  // first a[i] >= v
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (a[mid] < v) lo = mid + 1; else hi = mid;
  }
  return lo;
}
__device__ __forceinline__ int upper_bound_f(const float* a, int lo, int hi, float v) {  // first a[i] > v
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (a[mid] <= v) lo = mid + 1; else hi = mid;
  }
  return lo;
}

// [first, first + count) = the entries of the ascending array a[lo .. hi) inside [vlo, vhi]: lower_bound(vlo) and
// upper_bound(vhi) searched in ONE loop, so that the two chains of dependent loads travel together (these kernels are bound
// by the latency along a warp's serial chain, not by instruction count: profiles/r2_summary.md).
__device__ __forceinline__ int window_of(const float* a, int lo, int hi, float vlo, float vhi, int& first) {
  int l0 = lo, h0 = hi, l1 = lo, h1 = hi;
  while (l0 < h0 || l1 < h1) {
    const int m0 = (l0 + h0) >> 1, m1 = (l1 + h1) >> 1;
    const float k0 = a[min(m0, hi - 1)], k1 = a[min(m1, hi - 1)];
    if (l0 < h0) { if (k0 < vlo) l0 = m0 + 1; else h0 = m0; }
    if (l1 < h1) { if (k1 <= vhi) l1 = m1 + 1; else h1 = m1; }
  }
  first = l0;
  return max(l1 - l0, 0);
}

// M2 bounds |sinA| by thr(r_u) <= thr(r_max_upper); M1 (dot > 0) gives r_u > r_l.  The window
// shrinks as r_l grows, so evaluated at the smallest r of the layer's lower hits it covers them all.
// Returns the half width of the azimuth window around the lower hit, < 0 if nothing can pass.
__device__ __forceinline__ float md_window(const Cuts& c, int layer, float r_l, float r_max_upper) {
  if (!(r_max_upper > 0.0f) || !(r_max_upper * 1.000001f >= r_l)) return -1.0f;
  const float thr = fminf(1.0f, sin_threshold(c, r_max_upper, c.md_cos_eps[layer], c.md_sin_eps[layer]) * 1.00001f);
  const float d = delta_of(thr, fminf(1.0f, r_l / r_max_upper));
  return d * 1.001f + 2e-5f;
}

// S2 bounds |sinS| by thr(r_o); S4 on the inner MD bounds sinS * (ur_i / r_o) by sinA_i +- eps;
// S3 needs r_o > r_i.  [r_min_o, r_max_o] is the range of r of the anchors of the outer layer.
// Returns the window [dlo, dhi] of azimuth(outer) - azimuth(inner); dlo > dhi if nothing can pass.
__device__ __forceinline__ void seg_window(const Cuts& c, int layer, float r_i, float ur_i, float sinA_i,
                                           float r_min_o, float r_max_o, float& dlo, float& dhi) {
  dlo = 1.0f;
  dhi = -1.0f;
  if (!(r_max_o > r_i)) return;
  const float r_lo = fmaxf(r_min_o, r_i);
  float s_hi = fminf(1.0f, sin_threshold(c, r_max_o, c.seg_cos_eps, c.seg_sin_eps) * 1.00001f);
  float s_lo = -s_hi;
  if (ur_i > 0.0f && ur_i < 3.0e38f) {
    const float e = c.md_eps[layer] + 1e-5f;
    const float c_lo = (sinA_i - e) / ur_i, c_hi = (sinA_i + e) / ur_i;
    const float a = (c_lo >= 0.0f) ? c_lo * r_lo : c_lo * r_max_o;   // min over r_o of c_lo * r_o
    const float b = (c_hi >= 0.0f) ? c_hi * r_max_o : c_hi * r_lo;   // max over r_o of c_hi * r_o
    s_lo = fmaxf(s_lo, a - (1e-5f + 1e-5f * fabsf(a)));
    s_hi = fminf(s_hi, b + (1e-5f + 1e-5f * fabsf(b)));
  }
  if (!(s_lo <= s_hi)) return;
  const float q_lo = fminf(1.0f, r_i / r_lo), q_hi = r_i / r_max_o;
  // delta_of(s, q) falls with q for s > 0 and grows with q for s < 0 (d/dq = -s / sqrt(1 - q^2 s^2)): the extreme over
  // q in [q_hi, q_lo] sits at the end the sign of s names, one evaluation per bound
  const float hi = delta_of(s_hi, s_hi >= 0.0f ? q_hi : q_lo);
  const float lo = delta_of(s_lo, s_lo >= 0.0f ? q_lo : q_hi);
  dlo = lo - (3e-5f + 1e-3f * fabsf(lo));
  dhi = hi + (3e-5f + 1e-3f * fabsf(hi));
}

// Cheap necessary conditions for a window candidate, evaluated before the exact selection (which keeps the last
// word: whatever survives goes through seg_select).  With delta the azimuth of the outer anchor minus that of the
// inner one, the triangle (beam line, inner, outer) gives the cut variable of S2 / S4 in closed form,
//     sinS = r_o sin(delta) / sqrt(r_o^2 - 2 r_i r_o cos(delta) + r_i^2),
// here in fast arithmetic (|error| < 1e-5 from the rounding of delta, the cancellation in the denominator and the
// fast sin / cos / rsqrt / division); S4 on the OUTER mini-doublet and S3 are then tested with slack (2e-3 on a
// threshold of 0.057 / 0.092; 0.1 % + 0.5 mm on z0) that is orders of magnitude above that error.  On the PU200-like
// event 320 k window candidates -> 55.5 k segments: S3 rejects a third, S4-outer most of the rest.
__device__ __forceinline__ bool seg_prefilter(const Cuts& c, int layer_in, const float4& ai, const float4& ao,
                                              const float2& auxo, float delta) {
  // both tests are evaluated without a branch between them, so that the gathers of the outer record (anchor, aux) travel
  // together instead of the second waiting for the first test
  const float dr = ao.w - ai.w;
  const float z0 = ai.z - ai.w * __fdividef(ao.z - ai.z, dr);
  const bool s3_fails = fabsf(z0) > c.seg_z0_max[layer_in] * 1.001f + 0.05f;   // S3 (a NaN goes on to the exact test)
  float sd, cd;
  __sincosf(delta, &sd, &cd);
  const float den2 = (ao.w * ao.w + ai.w * ai.w) - 2.0f * ai.w * ao.w * cd;
  const float s = ao.w * sd * rsqrtf(den2);
  const float e2 = fabsf(auxo.y - s * __fdividef(auxo.x, ao.w));
  const bool s4_fails = den2 > 0.0f && e2 > c.md_eps[layer_in + 1] + 2e-3f;    // S4, outer mini-doublet
  return !(s3_fails | s4_fails);
}

__device__ __forceinline__ float r_min_of(const SlotHeader* h, int side, int layer) {
  return __int_as_float(0x7f800000 - h->r_min_inv[side][layer]);
}
__device__ __forceinline__ float r_max_of(const SlotHeader* h, int side, int layer) {
  return __int_as_float(h->r_max[side][layer]);
}

// ------------------------------------------------------------------------------------------
// a0: load + bin by (side, module) + order by azimuth + derive r
// blockIdx.y = event of the batch; its input arrays come from the pointer table `B`.
// Three launches.  The caller's arrays are read ONCE, by k_bin_count, which leaves a 28-byte record per hit; the other two
// kernels work from records.  The slot recycles itself: the last block of k_bin_count turns the bin counters into offsets,
// clears them for the next event and writes a fresh header; k_bin_scatter clears the look-back words on the side.
// ------------------------------------------------------------------------------------------
// Counters cnt[0 .. n] -> exclusive offsets start[0 .. n] (start[n] = total), counters cleared, by the whole block; the
// counters were incremented by other blocks (ld.cg).  Arrays are padded with zeros to a multiple of 4 ints (the slot layout
// rounds every array up to 256 bytes).  One block does this while the rest of the event's grid has retired, so what
// counts is its latency: a tile of NT x kPer int4 is loaded with all loads in flight at once.  Returns the total.
template <int NT, int kPer>
__device__ int block_offsets_from_counts(unsigned* cnt, unsigned* start, int n) {
  constexpr int W = NT / 32;
  __shared__ int warp_tot[W];
  __shared__ int s_carry;
  int4* c4 = reinterpret_cast<int4*>(cnt);
  int4* s4 = reinterpret_cast<int4*>(start);
  const int n4 = (n + 1 + 3) / 4;
  const int w = threadIdx.x >> 5, lane = (int)lane_id();
  if (threadIdx.x == 0) s_carry = 0;
  __syncthreads();
  for (int t0 = 0; t0 < n4; t0 += NT * kPer) {
    const int j0 = t0 + (int)threadIdx.x * kPer;
    int4 v[kPer];
#pragma unroll
    for (int k = 0; k < kPer; ++k) v[k] = (j0 + k < n4) ? __ldcg(c4 + j0 + k) : make_int4(0, 0, 0, 0);
    int mine = 0;
#pragma unroll
    for (int k = 0; k < kPer; ++k) mine += (v[k].x + v[k].y) + (v[k].z + v[k].w);
    const int incl = warp_incl_scan(mine);
    if (lane == 31) warp_tot[w] = incl;
    __syncthreads();
    int ex = s_carry + incl - mine, tile_total = 0;
#pragma unroll
    for (int i = 0; i < W; ++i) {
      const int t = warp_tot[i];
      ex += (i < w) ? t : 0;
      tile_total += t;
    }
#pragma unroll
    for (int k = 0; k < kPer; ++k) {
      if (j0 + k < n4) {
        s4[j0 + k] = make_int4(ex, ex + v[k].x, ex + v[k].x + v[k].y, ex + v[k].x + v[k].y + v[k].z);
        c4[j0 + k] = make_int4(0, 0, 0, 0);
      }
      ex += (v[k].x + v[k].y) + (v[k].z + v[k].w);
    }
    __syncthreads();
    if (threadIdx.x == 0) s_carry += tile_total;
    __syncthreads();
  }
  return s_carry;
}

// One pass over the caller's arrays -- the only one: per hit its azimuth key and, from the atomic on its (side, module)
// counter, its arrival rank in the bin, kept with the coordinates as a record (16 + 8 + 4 bytes: the key is stored twice,
// densely for the scatter and beside the coordinates for the final gather).  If the arrays are mapped host
// memory (in.stage) this pass IS the host-to-device copy: every array is read once over PCIe, coalesced.
// The block that finishes last in the event turns the counters into bin offsets (clearing them for the next event) and
// writes the header afresh: hit counts, dropped hits, every accumulator and ticket of the stage kernels at zero.
__global__ void __launch_bounds__(256) k_bin_count(const __grid_constant__ Params P, const __grid_constant__ HitBatch B) {
  Slot S(P, blockIdx.y);
  const HitInput& in = B.ev[blockIdx.y];
  SlotHeader* H = S.hdr();
  unsigned* cnt = S.bin_cnt();
  float4* rec4 = S.rec4();
  int2* recb = S.recb();
  float* reck = S.reck();
  const int nmod = P.L.n_modules;
  int bad = 0;
  for (int h = blockIdx.x * blockDim.x + threadIdx.x; h < in.n; h += gridDim.x * blockDim.x) {
    const int m = in.module[h];
    const unsigned sd = in.side[h];
    const float x = in.x[h], y = in.y[h], z = in.z[h];
    int bin = -1, rank = 0;
    float k = 0.0f;
    if (m < 0 || m >= nmod || sd > 1u) {
      ++bad;
    } else {
      const float2 cs = P.mod_cs[m];
      // azimuth relative to the module normal; non-finite hits (they can never pass a cut) go last
      k = atan2f(cs.x * y - cs.y * x, cs.x * x + cs.y * y);
      if (!(fabsf(k) <= 4.0f)) k = 3.0e38f;
      bin = (int)sd * nmod + m;
      rank = (int)atomicAdd(cnt + bin, 1u);
    }
    rec4[h] = make_float4(x, y, z, k);
    recb[h] = make_int2(bin, rank);
    reck[h] = k;
  }
  if (bad) atomicAdd(&H->bad_acc, (unsigned)bad);
  if (!last_block_done(&H->done[0], gridDim.x)) return;
  unsigned* start = S.bin_start();
  const int total = block_offsets_from_counts<256, 2>(cnt, start, P.L.n_bins);   // small tiles: the tail must not set the kernel's register count
  // fresh header: everything but the self-resetting tickets
  int* hw = reinterpret_cast<int*>(H);
  constexpr int kDone0 = offsetof(SlotHeader, done) / 4, kDone1 = offsetof(SlotHeader, ticket) / 4, kBad = offsetof(SlotHeader, bad_acc) / 4;
  for (int i = threadIdx.x; i < (int)(sizeof(SlotHeader) / 4); i += blockDim.x)
    if ((i < kDone0 || i >= kDone1) && i != kBad) hw[i] = 0;
  __syncthreads();
  if (threadIdx.x == 0) {
    H->n_hits = total;
    H->n_lower = (int)start[nmod];
    H->bad_hits = (int)H->bad_acc;
    H->bad_acc = 0;
  }
}

// Counters to offsets for the MD -> quintuplet incidence table of the cleaning stage: one block of 1024 threads per event.
__global__ void __launch_bounds__(1024) k_scan(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  block_scan_array4<1024, 3>(S.inc_start(), S.hdr()->n[LST_MD_]);
}

// (original index, key) of every hit to its (unsorted) place in its bin: bin offset + arrival rank -- no second atomic.
// On the side: the look-back words of the stage kernels are cleared for this event.
__global__ void __launch_bounds__(256) k_bin_scatter(const __grid_constant__ Params P, const __grid_constant__ HitBatch B) {
  Slot S(P, blockIdx.y);
  const int n = B.ev[blockIdx.y].n;
  const unsigned* start = S.bin_start();
  const int2* recb = S.recb();
  const float* reck = S.reck();
  int2* tki = S.tmp_ki();
  int* tbin = S.tmp_bin();
  const int tid = blockIdx.x * blockDim.x + threadIdx.x, nth = gridDim.x * blockDim.x;
  int4* lb = S.at<int4>(P.L.lb[0]);
  for (int i = tid; i < (int)(P.L.lb_bytes / 16); i += nth) lb[i] = make_int4(0, 0, 0, 0);
  for (int h = tid; h < n; h += nth) {
    const int2 b = recb[h];
    if (b.x < 0) continue;
    const unsigned pos = start[b.x] + (unsigned)b.y;
    tki[pos] = make_int2(h, (int)sortable_of(reck[h]));   // little endian: (index, key) = key in the high word
    tbin[pos] = b.x;
  }
}

// One thread per hit: its rank inside the bin by (key, original index) is the number of hits of the bin that come
// before it -- a loop over the bin (6 hits on average, all lanes busy whatever the bin sizes; neighbouring threads sit
// in the same or the next bin).  Then fetch the hit's record (one 16-byte gather), derive r, and keep the range of r per
// (side, layer) and the key range per module.
__global__ void __launch_bounds__(256) k_bin_order(const __grid_constant__ Params P) {
  __shared__ int s_rng[30];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int nmod = P.L.n_modules;
  if (threadIdx.x < 30) s_rng[threadIdx.x] = 0;
  __syncthreads();
  const int nh = H->n_hits;
  const unsigned* start = S.bin_start();
  const unsigned long long* tk = reinterpret_cast<const unsigned long long*>(S.tmp_ki());
  int* info = reinterpret_cast<int*>(S.mod_info());
  const int p = blockIdx.x * 256 + threadIdx.x;
  if (p < nh) {
    const int b = S.tmp_bin()[p];
    const int s = (int)start[b], e = (int)start[b + 1];
    const unsigned long long mine = tk[p];                   // (sortable key << 32) | original index
    const int orig = (int)(unsigned)mine;
    const float4 v = S.rec4()[orig];                         // (x, y, z, key)
    int rank = 0;
    {   // two entries per 16-byte load once the position is even (the array is 16-byte aligned)
      int j = s;
      if ((j & 1) && j < e) { rank += tk[j] < mine; ++j; }
      const ulonglong2* tk2 = reinterpret_cast<const ulonglong2*>(tk);
      for (; j + 1 < e; j += 2) {
        const ulonglong2 t = tk2[j >> 1];
        rank += (t.x < mine) + (t.y < mine);
      }
      if (j < e) rank += tk[j] < mine;
    }
    const int side = b >= nmod, m = b - side * nmod;
    const float r = sqrtf(v.x * v.x + v.y * v.y);
    const int dst = s + rank;
    S.hit4()[dst] = make_float4(v.x, v.y, v.z, r);
    S.hit_key()[dst] = v.w;
    S.hit_orig()[dst] = orig;
    S.hit_module()[dst] = m;
    if (!side) {
      if (rank == 0) info[4 * m + 2] = __float_as_int(v.w);
      if (rank == e - s - 1) info[4 * m + 3] = __float_as_int(v.w);
    }
    // range of r per (side, layer): neighbouring threads sit in the same or the next bin, so a warp
    // holds one or two (side, layer) groups -- one shared-memory atomic pair per group, not per hit
    const bool fin = r < 3.0e38f;
    const unsigned act = __ballot_sync(__activemask(), fin);
    if (fin) {
      const int layer = P.mod_layer[m], slot = side * 6 + layer;
      const unsigned grp = __match_any_sync(act, slot);
      const int rmax = __reduce_max_sync(grp, __float_as_int(r));
      const int rinv = __reduce_max_sync(grp, 0x7f800000 - __float_as_int(r));
      const int kabs = __reduce_max_sync(grp, __float_as_int(fabsf(v.w)));     // |key| <= 4: finite here
      if ((int)lane_id() == __ffs(grp) - 1) {
        atomicMax(&s_rng[slot], rinv);
        atomicMax(&s_rng[12 + slot], rmax);
        if (!side) atomicMax(&s_rng[24 + layer], kabs);      // the segment kernel bounds every module's key range by it
      }
    }
  }
  if (p < nmod && start[p + 1] == start[p]) {  // no lower hits: an empty key range
    info[4 * p + 2] = __float_as_int(3.0e38f);
    info[4 * p + 3] = __float_as_int(-3.0e38f);
  }
  // search space of the MD stage: sum over modules of (#lower hits) x (#upper hits)
  if (blockIdx.x * 256 < (unsigned)nmod) {
    unsigned long long c = 0;
    if (p < nmod) c = (unsigned long long)(start[p + 1] - start[p]) * (unsigned long long)(start[nmod + p + 1] - start[nmod + p]);
    c = warp_sum_ull(c);
    if (lane_id() == 0 && c) atomicAdd(&H->cand[LST_MD_], c);
  }
  __syncthreads();
  if (threadIdx.x < 30 && s_rng[threadIdx.x]) atomicMax(&H->r_min_inv[0][0] + threadIdx.x, s_rng[threadIdx.x]);   // r_min_inv, r_max, key_absmax
}

// ------------------------------------------------------------------------------------------
// the warp pipeline
// ------------------------------------------------------------------------------------------
// Flattened ranges: lane l owns `n` consecutive items starting at flat position `off` (exclusive
// scan of n over the warp).  For the tile of flat positions [tb, tb + 32) returns, for the lane at
// position tb + lane, the rank of its owner among the NON-EMPTY owners (index into a table of
// their lanes that the caller keeps).  Every non-empty owner that starts inside the tile sets the
// bit of its start; the owner of a position is the last start at or before it.
__device__ __forceinline__ int tile_owner(int n, int off, int tb) {
  const unsigned startbit = (n > 0 && off >= tb && off < tb + 32) ? (1u << (off - tb)) : 0u;
  const unsigned mask = __reduce_or_sync(kFull, startbit);
  const int before = __popc(__ballot_sync(kFull, n > 0 && off < tb));
  return before + __popc(mask & lanemask_le()) - 1;
}
// Table of the lanes of the non-empty owners, in order (tab[rank] = lane).
__device__ __forceinline__ void build_owner_table(int n, int* tab) {
  const unsigned ne = __ballot_sync(kFull, n > 0);
  if (n > 0) tab[__popc(ne & lanemask_lt())] = (int)lane_id();
  __syncwarp();
}

// single-pass ordered output: chunks of owners are handed out in order by a ticket; a warp
// learns where its chunk's objects start by decoupled look-back over the totals of the chunks
// before it (each chunk publishes its total as soon as it is known, so nothing waits on a
// warp that has not started).  status word: bits 63:62 = 1 total only, 2 = inclusive prefix.
__device__ __forceinline__ void st_status(unsigned long long* p, unsigned long long v) {
  asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long ld_status(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
// A chunk's total is published as soon as its walk is over (status 1 = total only), so no warp ever
// waits on another warp's look-back, only on its walk.
__device__ __forceinline__ void publish_aggregate(unsigned long long* status, int c, int total) {
  if (lane_id() == 0) st_status(status + c, ((c == 0 ? 2ull : 1ull) << 62) | (unsigned)total);
}
#ifndef LST_BACKOFF_MAX
#define LST_BACKOFF_MAX 32       // cap of the back-off in ns; same-box A/B of 32 / 128 / 1024 / 4096: 50.66 / 50.48 / 50.33 / 49.89 k events/s
#endif
// Called by all lanes of a warp, after publish_aggregate(c).  Returns the number of objects of
// chunks 0 .. c-1 and publishes chunk c's inclusive prefix (status 2).
__device__ __forceinline__ int resolve_base(unsigned long long* status, int c, int total) {
  if (c == 0) return 0;
  const int lane = (int)lane_id();
  int sum = 0;
  for (int j = c - 1;; j -= 32) {
    const int idx = j - lane;
    unsigned long long v = (idx >= 0) ? ld_status(status + idx) : (2ull << 62);
    unsigned ns = 32;
    while (__any_sync(kFull, (v >> 62) == 0)) {   // a predecessor is still walking: back off, do not burn issue slots
      __nanosleep(ns);
      if (ns < LST_BACKOFF_MAX) ns <<= 1;
      if ((v >> 62) == 0) v = ld_status(status + idx);
    }
    const unsigned pmask = __ballot_sync(kFull, (v >> 62) == 2);
    const int firstP = pmask ? __ffs(pmask) - 1 : 32;
    int contrib = (lane <= firstP) ? (int)(unsigned)(v & 0xffffffffull) : 0;
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) contrib += __shfl_xor_sync(kFull, contrib, d);
    sum += contrib;
    if (pmask) break;
  }
  if (lane == 0) st_status(status + c, (2ull << 62) | (unsigned)(sum + total));
  return sum;
}
// Next chunk of 32 owners of this warp.
__device__ __forceinline__ int warp_ticket(unsigned* ticket) {
  int c = 0;
  if (lane_id() == 0) c = (int)atomicAdd(ticket, 1u);
  return __shfl_sync(kFull, c, 0);
}

// a[lo .. hi) = v by one warp: 16-byte stores over the aligned middle (the arrays start on 256-byte boundaries).
__device__ __noinline__ void fill_ints(int* a, int lo, int hi, int v) {
  const int lane = (int)lane_id();
  const int mid0 = min((lo + 3) & ~3, hi), mid1 = max(hi & ~3, mid0);
  for (int i = lo + lane; i < mid0; i += 32) a[i] = v;
  int4* a4 = reinterpret_cast<int4*>(a);
  for (int i = (mid0 >> 2) + lane; i < (mid1 >> 2); i += 32) a4[i] = make_int4(v, v, v, v);
  for (int i = mid1 + lane; i < hi; i += 32) a[i] = v;
}

#ifndef LST_MD_BLOCKS
#define LST_MD_BLOCKS 6          // resident blocks per SM the launch bounds ask for (A/B of round 2: profiles/r2_summary.md)
#endif
#ifndef LST_T5_BLOCKS
#define LST_T5_BLOCKS 4
#endif
constexpr int kWarps = 8;        // warps per block of the MD / T3 / T5 kernels
constexpr int kSegWarps = 4;     // of the segment kernel (more shared memory per warp)
constexpr int kQueue = 64;       // queue slots per warp (a push adds <= 32, a drain starts at >= 32)

// ------------------------------------------------------------------------------------------
// a1: mini-doublets.  Owner = lower hit; its candidates are the upper hits of the same module
// inside the azimuth window (two binary searches in the key-ordered upper bin).
// ------------------------------------------------------------------------------------------
constexpr int kMdStash = 96;
struct MdWarp {
  float4 lo[32];
  int layer[32], tab[32];
  int cnt[2][32];               // objects per owner, of the chunk being walked / the chunk awaiting its base
  int stI[2][kMdStash];
  float stS[2][kMdStash];
};

// i = index of the lower hit (owner), u = index of the upper hit.
__device__ __forceinline__ void md_emit(const Params& P, const Slot& S, int pos, int i, int u, float sinA) {
  if (pos >= P.L.cap_md) return;
  // all gathers first (a store that needs a loaded value holds up the loads behind it), then the stores
  const float4 lo = S.hit4()[i], up = S.hit4()[u];
  const float key = S.hit_key()[i];
  const int orig_lo = S.hit_orig()[i], orig_up = S.hit_orig()[u], module = S.hit_module()[i];
  const float dx = up.x - lo.x, dy = up.y - lo.y;
  const float cross = lo.x * dy - lo.y * dx, dot = lo.x * dx + lo.y * dy;   // as in md_select
  const float dphi = atan2f(lo.x * up.y - lo.y * up.x, lo.x * up.x + lo.y * up.y), dphichange = atan2f(cross, dot);
  S.md_anchor()[pos] = lo;
  S.md_aux()[pos] = make_float2(up.w, sinA);
  S.md_key()[pos] = key;
  S.md_hits()[pos] = make_int2(orig_lo, orig_up);
  if (P.store_half) reinterpret_cast<__half2*>(S.md_out())[pos] = __floats2half2_rn(dphi, dphichange);   // [H]
  else S.md_out()[pos] = make_float2(dphi, dphichange);
  S.md_module()[pos] = module;
}

template <bool DIRECT>
__device__ __forceinline__ int md_walk(const Params& P, const Slot& S, MdWarp& sh, int buf, int n, int off, int total,
                                       int j0, int i0, int base) {
  const float4* hit4 = S.hit4();
  const int lane = (int)lane_id();
  int running = 0;
  for (int tb = 0; tb < total; tb += 32) {
    const int rk = tile_owner(n, off, tb);
    const int j = tb + lane;
    const int ol = (j < total) ? sh.tab[rk] : 0;
    const int ooff = __shfl_sync(kFull, off, ol), oj0 = __shfl_sync(kFull, j0, ol);
    bool pass = false;
    MdOut o;
    int u = 0;
    if (j < total) {
      u = oj0 + (j - ooff);
      pass = md_select(P.cuts, sh.layer[ol], sh.lo[ol], hit4[u], o);
    }
    const unsigned bal = __ballot_sync(kFull, pass);
    if (pass) {
      const int pos = running + __popc(bal & lanemask_lt());
      if (!DIRECT) {
        atomicAdd(&sh.cnt[buf][ol], 1);
        if (pos < kMdStash) { sh.stI[buf][pos] = (ol << 26) | u; sh.stS[buf][pos] = o.sinA; }
      } else {
        md_emit(P, S, base + pos, i0 + ol, u, o.sinA);
      }
    }
    running += __popc(bal);
  }
  return running;
}

__global__ void __launch_bounds__(kWarps * 32, LST_MD_BLOCKS) k_md(const __grid_constant__ Params P) {
  __shared__ MdWarp shw[kWarps];
  __shared__ float s_w[6], s_rmaxU[6];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int nmod = P.L.n_modules, cap = P.L.cap_md;
  const int nLower = H->n_lower;
  const int nChunks = (nLower + kChunk - 1) / kChunk;
  const int lane = (int)lane_id();
  MdWarp& sh = shw[threadIdx.x >> 5];
  if (threadIdx.x < 6) {
    const float ru = r_max_of(H, 1, threadIdx.x);
    s_rmaxU[threadIdx.x] = ru;
    s_w[threadIdx.x] = md_window(P.cuts, threadIdx.x, r_min_of(H, 0, threadIdx.x), ru);
  }
  __syncthreads();
  const unsigned* bs = S.bin_start();
  const float* hkey = S.hit_key();
  const int* hmod = S.hit_module();
  int* md_start = S.md_start();
  int* info = reinterpret_cast<int*>(S.mod_info());
  unsigned long long* status = S.lb(LST_MD_);
  unsigned long long evals = 0;

  // writes what depends on the chunk's base: per-module tables, the grand total (+ the objects
  // themselves when they sit in the stash)
  auto finish = [&](int C, int b, int total, int base, bool from_stash) {
    const int i0 = C * kChunk, i = i0 + lane;
    if (from_stash)
      for (int t = lane; t < total; t += 32) {
        const int v = sh.stI[b][t];
        md_emit(P, S, base + t, i0 + (int)((unsigned)v >> 26), v & (kMaxCap - 1), sh.stS[b][t]);
      }
    int tot;
    const int first = min(base + warp_excl_scan(sh.cnt[b][lane], tot), cap);
    if (i < nLower) {
      // module table: the first lower hit of a module (and the modules without lower hits before it)
      const int m = hmod[i], m_prev = (i > 0) ? hmod[i - 1] : -1;
      for (int mm = m_prev + 1; mm <= m; ++mm) {
        md_start[mm] = first;
        info[4 * mm] = first;
        if (mm > 0) info[4 * (mm - 1) + 1] = first;
      }
      if (i == nLower - 1) {
        const int end = min(base + total, cap);
        for (int mm = m + 1; mm <= nmod; ++mm) {
          md_start[mm] = end;
          if (mm < nmod) info[4 * mm] = end;
          info[4 * (mm - 1) + 1] = end;
        }
        publish_total(H, LST_MD_, base + total, cap);
      }
    }
    __syncwarp();
  };

  int buf = 0, pC = -1, pTotal = 0;   // pC: chunk whose objects wait in stash[buf ^ 1] for their base
  for (;;) {
    const int C = warp_ticket(&H->ticket[LST_MD_]);
    if (C >= nChunks) {
      if (C == 0) {  // no lower hits at all: the first ticket publishes the empty result
        for (int m = lane; m <= nmod; m += 32) {
          md_start[m] = 0;
          if (m < nmod) { info[4 * m] = 0; info[4 * m + 1] = 0; }
        }
        if (lane == 0) publish_total(H, LST_MD_, 0, cap);
      }
      break;
    }
    const int i0 = C * kChunk, i = i0 + lane;
    int n = 0, j0 = 0;
    if (i < nLower) {
      const int m = hmod[i];
      const int layer = P.mod_layer[m];
      const int u0 = (int)bs[nmod + m], u1 = (int)bs[nmod + m + 1];
      const float4 lo = S.hit4()[i];
      const float kl = hkey[i];
      sh.lo[lane] = lo;
      sh.layer[lane] = layer;
      const float w = s_w[layer];
      if (u1 > u0 && w >= 0.0f && s_rmaxU[layer] * 1.000001f >= lo.w) {
        j0 = u0;
        n = u1 - u0;
        if (fabsf(kl) + w < 1.5f) n = window_of(hkey, u0, u1, kl - w, kl + w, j0);
      }
    }
    sh.cnt[buf][lane] = 0;
    evals += (unsigned long long)n;
    int total_c;
    const int off = warp_excl_scan(n, total_c);
    build_owner_table(n, sh.tab);
    const int total = md_walk<false>(P, S, sh, buf, n, off, total_c, j0, i0, 0);
    publish_aggregate(status, C, total);
    __syncwarp();
    if (pC >= 0) {   // the previous chunk has had a whole walk of slack: its base is (almost always) there
      finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
      pC = -1;
    }
    if (total <= kMdStash) {
      pC = C; pTotal = total; buf ^= 1;
    } else {           // does not fit the stash: resolve now and walk again, writing directly
      if (lane == 0) atomicAdd(&H->rewalk[LST_MD_], 1ull);
      const int base = resolve_base(status, C, total);
      md_walk<true>(P, S, sh, buf, n, off, total_c, j0, i0, base);
      finish(C, buf, total, base, false);
    }
  }
  if (pC >= 0) finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
  evals = warp_sum_ull(evals);
  if (lane == 0 && evals) atomicAdd(&H->eval[LST_MD_], evals);
}

// ------------------------------------------------------------------------------------------
// a2: segments.  Owner = inner MD.  Three levels, each compacted before the next:
//   A  lane = inner MD; the (inner MD, connected module) pairs of the part of the map row the MD's
//      window can reach (rows are ordered by azimuth offset: one run, found by a search): module
//      has MDs and its key range meets the MD's azimuth window?         -> pair queue
//   B  surviving pairs: window of outer MDs by a search (both bounds in one loop) in the module's
//      key-ordered MD list; the windows are flattened into candidates, closed-form pre-filter
//                                                                        -> candidate queue
//   C  candidates, 32 at a time: the SPEC selection                     -> stash (arrival order + rank)
// Segments come out ordered by (inner MD, outer MD): placed by (owner, arrival rank), then every
// owner's few segments are put in ascending outer MD.
// ------------------------------------------------------------------------------------------
// The block's shared memory decides how much of the SM's 256 KB is left as L1: 7 resident blocks must stay within the 196 KB
// carve-out (27 648 B per block incl. the 1 KB the system reserves), or the next carve-out (228 KB) halves the L1 and costs 5 %
// (measured: 48.1 k against 50.5 k events/s for 1.3 KB more per block).  Smaller stashes for a smaller carve-out lose to the
// re-walks they cause (kSegStash 104: 47.8 k).
constexpr int kSegStash = 152;
struct SegWarp {
  float4 a4[32];
  float2 aux[32];
  float key[32], dlo[32], dhi[32];
  int layer[32], tab[32], ptab[32];
  int2 pq[kQueue], cq[kQueue];
  int cnt[2][32];
  int stI[2][kSegStash];
  float2 stV[2][kSegStash];
  unsigned char stR[2][kSegStash];   // rank of a stashed segment among its owner's
};
static_assert(kSegWarps * sizeof(SegWarp) + 64 + 1024 <= 28672, "k_seg: 7 blocks per SM must fit the 196 KB shared-memory carve-out");

// i / o = index of the inner / outer MD.
__device__ __forceinline__ void seg_emit(const Params& P, const Slot& S, int pos, int i, int o, float sinS, float z0) {
  if (pos >= P.L.cap_seg) return;
  const float4 ai = S.md_anchor()[i], ao = S.md_anchor()[o];
  const float dx = ao.x - ai.x, dy = ao.y - ai.y;
  const float cross = ai.x * dy - ai.y * dx, dot = ai.x * dx + ai.y * dy;   // as in seg_select
  S.seg_md()[pos] = make_int2(i, o);
  const float dphi = atan2f(ai.x * ao.y - ai.y * ao.x, ai.x * ao.x + ai.y * ao.y), dphichange = atan2f(cross, dot);
  if (P.store_half) {   // [H]
    const __half2 a = __floats2half2_rn(sinS, z0), b = __floats2half2_rn(dphi, dphichange);
    reinterpret_cast<uint2*>(S.seg_f())[pos] = make_uint2(*reinterpret_cast<const unsigned*>(&a), *reinterpret_cast<const unsigned*>(&b));
  } else {
    S.seg_f()[pos] = make_float4(sinS, z0, dphi, dphichange);
  }
}

// Level A: lane = inner MD of the chunk, and the warp steps through the rows of the module map in lockstep (entry t of every
// lane's row in iteration t; mini-doublets of one module read the same row entry: one broadcast load).  The (MD, connected
// module) pairs are not flattened, so there is no owner lookup per pair (the flattened form of round 1 spent a third of the
// kernel's instructions in level A; same-box A/B 50.5 k -> 51.1 k events/s).  Pairs reach the queues ordered by (row entry, MD);
// for ONE inner MD they still arrive in ascending outer MD (rows ascend, the queues are FIFO), so a segment's place among its
// owner's is the number of that owner's segments seen before it (`rank`), and its CSR position is
// base + (segments of the lanes before the owner) + rank.  cnt[cb] counts per owner as the walk goes.
template <bool DIRECT>
__device__ __forceinline__ int seg_walk(const Params& P, const Slot& S, SegWarp& sh, int buf, int nt, int row0, int i0,
                                        int base, unsigned long long& evals_acc) {
  const float4* anchor = S.md_anchor();
  const float2* aux = S.md_aux();
  const float* mkey = S.md_key();
  const int4* mod_info = S.mod_info();
  const int lane = (int)lane_id();
  const int cb = DIRECT ? buf ^ 1 : buf;   // running per-owner counters (the direct walk keeps the first walk's totals in cnt[buf])
  // windows evaluated in this walk: 32 bits suffice (at most 64 x the mini-doublets of the event per lane, capacities are
  // below 2^26), the 64-bit total stays out of the loops
  unsigned evals = 0;
  int running = 0;
  int ph = 0, pt = 0, ch = 0, ct = 0;

  auto levelC = [&](bool valid, int2 it) {
    bool pass = false;
    SegOut so;
    const int ol = it.x, o = it.y;
    if (valid) pass = seg_select(P.cuts, sh.layer[ol], sh.a4[ol], sh.aux[ol], anchor[o], aux[o], so);
    const unsigned bal = __ballot_sync(kFull, pass);
    if (bal) {
      unsigned grp = 0;
      int rank = 0;
      if (pass) {
        grp = __match_any_sync(bal, ol);
        rank = sh.cnt[cb][ol] + __popc(grp & lanemask_lt());
        if (!DIRECT) {
          const int pos = running + __popc(bal & lanemask_lt());
          if (pos < kSegStash) {
            sh.stI[buf][pos] = (ol << 26) | o; sh.stV[buf][pos] = make_float2(so.sinS, so.z0);
            sh.stR[buf][pos] = (unsigned char)rank;
          }
        } else {
          seg_emit(P, S, base + sh.tab[ol] + rank, i0 + ol, o, so.sinS, so.z0);
        }
      }
      __syncwarp();
      if (pass && (grp & lanemask_lt()) == 0) sh.cnt[cb][ol] += __popc(grp);
      running += __popc(bal);
    }
  };
  auto drainC = [&](bool all) {
    while (ct - ch >= 32 || (all && ct > ch)) {
      __syncwarp();
      const bool valid = lane < ct - ch;
      int2 it = make_int2(0, 0);
      if (valid) it = sh.cq[(ch + lane) & (kQueue - 1)];
      levelC(valid, it);
      ch += min(32, ct - ch);
      __syncwarp();
    }
  };
  auto levelB = [&](bool valid, int2 it) {
    int first = 0, cnt = 0;
    const int ol = (int)((unsigned)it.x >> 26);
    if (valid) {
      const int4 info = mod_info[it.x & (kMaxCap - 1)];
      const float c0 = __int_as_float(it.y), dlo = sh.dlo[ol], dhi = sh.dhi[ol];
      if (!(fabsf(c0) + fmaxf(fabsf(dlo), fabsf(dhi)) < 3.0f)) {
        first = info.x;  // azimuth wrap possible (never with a sane geometry): no window
        cnt = info.y - info.x;
      } else {
        cnt = window_of(mkey, info.x, info.y, c0 + dlo, c0 + dhi, first);
      }
    }
    if (!DIRECT) evals += (unsigned)cnt;
    int nc;
    const int coff = warp_excl_scan(cnt, nc);
    build_owner_table(cnt, sh.ptab);
    const float c0v = __int_as_float(it.y);
    for (int tb = 0; tb < nc; tb += 32) {
      const int rk = tile_owner(cnt, coff, tb);
      const int j = tb + lane;
      const int pl = (j < nc) ? sh.ptab[rk] : 0;
      const int o = __shfl_sync(kFull, first, pl) + (j - __shfl_sync(kFull, coff, pl));
      const int iol = __shfl_sync(kFull, ol, pl);
      const float c0p = __shfl_sync(kFull, c0v, pl);
      bool keep = false;
      if (j < nc) keep = seg_prefilter(P.cuts, sh.layer[iol], sh.a4[iol], anchor[o], aux[o], mkey[o] - c0p);
      const unsigned bal = __ballot_sync(kFull, keep);
      if (keep) sh.cq[(ct + __popc(bal & lanemask_lt())) & (kQueue - 1)] = make_int2(iol, o);
      ct += __popc(bal);
      drainC(false);
    }
    __syncwarp();
  };
  auto drainB = [&](bool all) {
    while (pt - ph >= 32 || (all && pt > ph)) {
      __syncwarp();
      const bool valid = lane < pt - ph;
      int2 it = make_int2(0, 0);
      if (valid) it = sh.pq[(ph + lane) & (kQueue - 1)];
      levelB(valid, it);
      ph += min(32, pt - ph);
      __syncwarp();
    }
  };
  // A: row entry t of every lane; the entry after it is fetched (target, azimuth offset, the target's module record) before
  // this one is tested
  struct AEntry {
    int tgt;
    float dphi;
    int4 info;
  };
  auto loadA = [&](int t) {
    AEntry e;
    e.tgt = 0;
    e.dphi = 0.0f;
    e.info = make_int4(0, 0, 0, 0);
    if (t < nt) {
      // the direct walk reads the row in ascending target order: its segments arrive in CSR order
      e.tgt = (DIRECT ? P.map_targets_asc : P.map_targets)[row0 + t];
      e.dphi = (DIRECT ? P.map_dphi_asc : P.map_dphi)[row0 + t];
      e.info = mod_info[e.tgt];
    }
    return e;
  };
  const int max_nt = __reduce_max_sync(kFull, nt);
  AEntry cur = loadA(0);
  for (int t = 0; t < max_nt; ++t) {

    // no branches (an entry beyond the lane's run is all zeros: an empty module)
    const int4 info = cur.info;
    const float dlo = sh.dlo[lane], dhi = sh.dhi[lane];
    const float c0 = sh.key[lane] + cur.dphi;
    const bool wrap = !(fabsf(c0) + fmaxf(fabsf(dlo), fabsf(dhi)) < 3.0f);
    const bool meets = (c0 + dhi >= __int_as_float(info.z)) & (c0 + dlo <= __int_as_float(info.w));
    const bool keep = (t < nt) & (info.y > info.x) & (dlo <= dhi) & (wrap | meets);
    const unsigned bal = __ballot_sync(kFull, keep);
    if (keep) sh.pq[(pt + __popc(bal & lanemask_lt())) & (kQueue - 1)] = make_int2((lane << 26) | cur.tgt, __float_as_int(c0));
    pt += __popc(bal);
    drainB(false);
    cur = loadA(t + 1);   // (fetching it before this entry is tested was measured: the registers it holds cost more, 50.2 k)
  }
  drainB(true);
  drainC(true);
  evals_acc += evals;
  return running;
}

__global__ void __launch_bounds__(kSegWarps * 32, 7) k_seg(const __grid_constant__ Params P) {
  __shared__ SegWarp shw[kSegWarps];
  __shared__ float s_rMinO[6], s_rMaxO[6];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int cap = P.L.cap_seg;
  const int nAll = H->n[LST_MD_];
  // mini-doublets of the outermost layer have no map row: with module ids ordered by layer (P.live_modules[2] = leading modules
  // on layers 0..4) they are the tail of the MD list; only the MDs before it are walked
  int nMD = nAll;
  if (P.live_modules[2] < P.L.n_modules && !H->overflow) nMD = min(nAll, S.md_start()[P.live_modules[2]]);
  const int nChunks = (nMD + kChunk - 1) / kChunk;
  const int lane = (int)lane_id();
  SegWarp& sh = shw[threadIdx.x >> 5];
  __shared__ float s_keyMax[6];
  if (threadIdx.x < 6) {
    s_rMinO[threadIdx.x] = r_min_of(H, 0, threadIdx.x);
    s_rMaxO[threadIdx.x] = r_max_of(H, 0, threadIdx.x);
    s_keyMax[threadIdx.x] = __int_as_float(H->key_absmax[threadIdx.x]);   // every module's key range lies within +- this
  }
  __syncthreads();
  int* seg_start = S.seg_start();
  unsigned long long* status = S.lb(LST_SEG_);
  unsigned long long evals = 0;
  {
    // The method's search space (lst_stats.candidates): every pair of an MD with an MD of a connected module, summed per
    // MODULE here (MDs of a module x MDs of its row), a slice of the modules per block -- the walk below only looks at the
    // part of a row an MD's window can reach and cannot count it.
    const int* md_start = S.md_start();
    const int4* mod_info = S.mod_info();
    unsigned long long space = 0;
    for (int m = blockIdx.x * blockDim.x + threadIdx.x; m < P.L.n_modules; m += gridDim.x * blockDim.x) {
      const int n_in = md_start[m + 1] - md_start[m];
      if (n_in <= 0) continue;
      int n_out = 0;
      for (int e = P.map_offsets[m]; e < P.map_offsets[m + 1]; ++e) {
        const int4 info = mod_info[P.map_targets[e]];
        n_out += info.y - info.x;
      }
      space += (unsigned long long)n_in * (unsigned long long)n_out;
    }
    space = warp_sum_ull(space);
    if (lane == 0 && space) atomicAdd(&H->cand[LST_SEG_], space);
  }

  auto finish = [&](int C, int b, int total, int base, bool from_stash) {
    const int i0 = C * kChunk, i = i0 + lane;
    int tot;
    const int ex = warp_excl_scan(sh.cnt[b][lane], tot);
    if (from_stash) {   // the stash is in arrival order: place by (owner, rank)
      sh.tab[lane] = ex;
      __syncwarp();
    }
    if (from_stash)
      for (int t = lane; t < total; t += 32) {
        const int v = sh.stI[b][t];
        const float2 f = sh.stV[b][t];
        const int ol = (int)((unsigned)v >> 26);
        seg_emit(P, S, base + sh.tab[ol] + sh.stR[b][t], i0 + ol, v & (kMaxCap - 1), f.x, f.y);
      }
    // An owner's segments were found in the order of its row (by azimuth offset), not by outer MD: the owner lane puts its
    // one to three segments in ascending outer MD (insertion sort of the stored records; the other lanes' stores first).
    // A chunk written by the direct walk is in order already (it reads the rows by ascending target).
    __syncwarp();
    if (from_stash) {
      const int mine = sh.cnt[b][lane];
      const int lo = min(base + ex, cap), hi = min(base + ex + mine, cap);
      int2* smd = S.seg_md();
      for (int k = lo + 1; k < hi; ++k) {
        const int2 key = smd[k];
        if (smd[k - 1].y <= key.y) continue;
        if (P.store_half) {
          uint2* sf = reinterpret_cast<uint2*>(S.seg_f());
          const uint2 val = sf[k];
          int j = k - 1;
          for (; j >= lo && smd[j].y > key.y; --j) { smd[j + 1] = smd[j]; sf[j + 1] = sf[j]; }
          smd[j + 1] = key; sf[j + 1] = val;
        } else {
          float4* sf = S.seg_f();
          const float4 val = sf[k];
          int j = k - 1;
          for (; j >= lo && smd[j].y > key.y; --j) { smd[j + 1] = smd[j]; sf[j + 1] = sf[j]; }
          smd[j + 1] = key; sf[j + 1] = val;
        }
      }
    }
    if (i < nMD) seg_start[i] = min(base + ex, cap);
    if (i0 + 31 >= nMD - 1) {
      fill_ints(seg_start, nMD, nAll + 1, min(base + total, cap));
      if (i == nMD - 1) publish_total(H, LST_SEG_, base + total, cap);
    }
    __syncwarp();
  };

  int buf = 0, pC = -1, pTotal = 0;
  for (;;) {
    const int C = warp_ticket(&H->ticket[LST_SEG_]);
    if (C >= nChunks) {
      if (C == 0) {  // no MDs with a map row at all: the first ticket publishes the empty result
        fill_ints(seg_start, 0, nAll + 1, 0);
        if (lane == 0) publish_total(H, LST_SEG_, 0, cap);
      }
      break;
    }
    const int i0 = C * kChunk, i = i0 + lane;
    int nt = 0, row0 = 0;
    if (i < nMD) {
      const float4 a = S.md_anchor()[i];
      const float2 x = S.md_aux()[i];
      const int A = S.md_module()[i];
      row0 = P.map_offsets[A];
      nt = P.map_offsets[A + 1] - row0;
      const int layer = P.mod_layer[A];
      const float key = S.md_key()[i];
      float dlo = 1.0f, dhi = -1.0f;
      if (nt > 0) seg_window(P.cuts, layer, a.w, x.x, x.y, s_rMinO[layer + 1], s_rMaxO[layer + 1], dlo, dhi);
      if (!(dlo <= dhi)) {
        nt = 0;
      } else if (nt > 0) {
        // The part of the row this MD can reach.  A connected module's key range lies within +-W (the largest |key| of the
        // outer layer's hits), and level A needs key + offset + dhi >= kmin and key + offset + dlo <= kmax, so the offset
        // lies in [-W - key - dhi, W - key - dlo]: one run of the row, which is ordered by offset (1e-4 rad of slack
        // against the rounding of these sums).  Where an azimuth wrap is possible the whole row stays.
        const float W = s_keyMax[layer + 1];
        if (W + fabsf(key) + fmaxf(fabsf(dlo), fabsf(dhi)) < 1.5f) {
          int t0;
          nt = window_of(P.map_dphi, row0, row0 + nt, (-W - key - dhi) - 1e-4f, (W - key - dlo) + 1e-4f, t0);
          row0 = t0;
        }
      }
      sh.a4[lane] = a;
      sh.aux[lane] = x;
      sh.key[lane] = key;
      sh.dlo[lane] = dlo;
      sh.dhi[lane] = dhi;
      sh.layer[lane] = layer;
    }
    sh.cnt[buf][lane] = 0;
    __syncwarp();
    const int total = seg_walk<false>(P, S, sh, buf, nt, row0, i0, 0, evals);
    publish_aggregate(status, C, total);
    __syncwarp();
    if (pC >= 0) {
      finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
      pC = -1;
    }
    if (total <= kSegStash) {
      pC = C; pTotal = total; buf ^= 1;
    } else {
      if (lane == 0) atomicAdd(&H->rewalk[LST_SEG_], 1ull);
      const int base = resolve_base(status, C, total);
      int tot;   // per-owner offsets from the first walk's totals; fresh running counters
      sh.tab[lane] = warp_excl_scan(sh.cnt[buf][lane], tot);
      sh.cnt[buf ^ 1][lane] = 0;
      __syncwarp();
      // over the WHOLE row in ascending target order (the reachable run is a run of the row ordered by azimuth offset only):
      // an owner's segments then arrive by ascending outer MD and need no sort -- a chunk of a dense event holds thousands
      int nt_all = 0, row_all = 0;
      if (i < nMD && nt > 0) {
        const int A = S.md_module()[i];
        row_all = P.map_offsets[A];
        nt_all = P.map_offsets[A + 1] - row_all;
      }
      seg_walk<true>(P, S, sh, buf, nt_all, row_all, i0, base, evals);
      finish(C, buf, total, base, false);
    }
  }
  if (pC >= 0) finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
  evals = warp_sum_ull(evals);
  if (lane == 0 && evals) atomicAdd(&H->eval[LST_SEG_], evals);
}

// ------------------------------------------------------------------------------------------
// a3: triplets.  Owner = first segment a = (m1, m2); candidates are the segments leaving m2, a
// contiguous range because segments are stored by inner MD.
// ------------------------------------------------------------------------------------------
constexpr int kT3Stash = 96;
struct T3Warp {
  float4 p1[32], p2[32];
  int layer[32], tab[32];
  int cnt[2][32];
  int stI[2][kT3Stash];
  float2 stV[2][kT3Stash];
};

// a / b = index of the first / second segment.
__device__ __forceinline__ void t3_emit(const Params& P, const Slot& S, int pos, int a, int b, float kappa, float chi2) {
  if (pos >= P.L.cap_t3) return;
  const int2 ma = S.seg_md()[a], mb = S.seg_md()[b];
  S.t3_pack()[pos] = make_int4(ma.x, ma.y, mb.y, __float_as_int(kappa));
  S.t3_seg()[pos] = make_int2(a, b);
  if (P.store_half) reinterpret_cast<__half*>(S.t3_chi2())[pos] = __float2half_rn(chi2);   // [H]
  else S.t3_chi2()[pos] = chi2;
}

template <bool DIRECT>
__device__ __forceinline__ int t3_walk(const Params& P, const Slot& S, T3Warp& sh, int buf, int n, int off, int total,
                                       int b0, int a0, int base) {
  const int2* seg_md = S.seg_md();
  const float4* anchor = S.md_anchor();
  const int lane = (int)lane_id();
  int running = 0;
  for (int tb = 0; tb < total; tb += 32) {
    const int rk = tile_owner(n, off, tb);
    const int j = tb + lane;
    const int ol = (j < total) ? sh.tab[rk] : 0;
    const int b = __shfl_sync(kFull, b0, ol) + (j - __shfl_sync(kFull, off, ol));
    bool pass = false;
    float kappa = 0.0f, chi2 = 0.0f;
    if (j < total) pass = t3_select(P.cuts, sh.layer[ol], sh.p1[ol], sh.p2[ol], anchor[seg_md[b].y], kappa, chi2);
    const unsigned bal = __ballot_sync(kFull, pass);
    if (pass) {
      const int pos = running + __popc(bal & lanemask_lt());
      if (!DIRECT) {
        atomicAdd(&sh.cnt[buf][ol], 1);
        if (pos < kT3Stash) { sh.stI[buf][pos] = (ol << 26) | b; sh.stV[buf][pos] = make_float2(kappa, chi2); }
      } else {
        t3_emit(P, S, base + pos, a0 + ol, b, kappa, chi2);
      }
    }
    running += __popc(bal);
  }
  return running;
}

__global__ void __launch_bounds__(kWarps * 32, 6) k_t3(const __grid_constant__ Params P) {
  __shared__ T3Warp shw[kWarps];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int cap = P.L.cap_t3;
  const int nAll = H->n[LST_SEG_];
  // segments whose inner MD sits on layer 4 cannot start a triplet; with module ids ordered by layer they are the tail of the
  // segment list (P.live_modules[1] = leading modules on layers 0..3): only the segments before it are walked, the CSR entries
  // of the rest are filled in by the warp of the last chunk
  int nSeg = nAll;
  if (P.live_modules[1] < P.L.n_modules && !H->overflow) nSeg = min(nAll, S.seg_start()[S.md_start()[P.live_modules[1]]]);
  const int nChunks = (nSeg + kChunk - 1) / kChunk;
  const int lane = (int)lane_id();
  T3Warp& sh = shw[threadIdx.x >> 5];
  const int* seg_start = S.seg_start();
  int* t3_start = S.t3_start();
  unsigned long long* status = S.lb(LST_T3_);
  unsigned long long cand = 0;

  auto finish = [&](int C, int b, int total, int base, bool from_stash) {
    const int a0 = C * kChunk, a = a0 + lane;
    if (from_stash)
      for (int t = lane; t < total; t += 32) {
        const int v = sh.stI[b][t];
        const float2 f = sh.stV[b][t];
        t3_emit(P, S, base + t, a0 + (int)((unsigned)v >> 26), v & (kMaxCap - 1), f.x, f.y);
      }
    int tot;
    const int ex = warp_excl_scan(sh.cnt[b][lane], tot);
    if (a < nSeg) t3_start[a] = min(base + ex, cap);
    if (a0 + 31 >= nSeg - 1) {
      fill_ints(t3_start, nSeg, nAll + 1, min(base + total, cap));
      if (a == nSeg - 1) publish_total(H, LST_T3_, base + total, cap);
    }
    __syncwarp();
  };

  int buf = 0, pC = -1, pTotal = 0;
  for (;;) {
    const int C = warp_ticket(&H->ticket[LST_T3_]);
    if (C >= nChunks) {
      if (C == 0) {
        fill_ints(t3_start, 0, nAll + 1, 0);
        if (lane == 0) publish_total(H, LST_T3_, 0, cap);
      }
      break;
    }
    const int a0 = C * kChunk, a = a0 + lane;
    int n = 0, b0 = 0;
    if (a < nSeg) {
      // every load of the owner's record is issued before any is needed (also for owners that turn out to have no
      // candidates): the chains travel together
      const int2 ma = S.seg_md()[a];
      const int s0 = seg_start[ma.y], s1 = seg_start[ma.y + 1];
      const float4 p1 = S.md_anchor()[ma.x], p2 = S.md_anchor()[ma.y];
      const int layer = P.mod_layer[S.md_module()[ma.x]];
      b0 = s0;
      n = s1 - s0;
      sh.p1[lane] = p1;
      sh.p2[lane] = p2;
      sh.layer[lane] = layer;
    }
    sh.cnt[buf][lane] = 0;
    cand += (unsigned long long)n;
    int total_c;
    const int off = warp_excl_scan(n, total_c);
    build_owner_table(n, sh.tab);
    const int total = t3_walk<false>(P, S, sh, buf, n, off, total_c, b0, a0, 0);
    publish_aggregate(status, C, total);
    __syncwarp();
    if (pC >= 0) {
      finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
      pC = -1;
    }
    if (total <= kT3Stash) {
      pC = C; pTotal = total; buf ^= 1;
    } else {
      if (lane == 0) atomicAdd(&H->rewalk[LST_T3_], 1ull);
      const int base = resolve_base(status, C, total);
      t3_walk<true>(P, S, sh, buf, n, off, total_c, b0, a0, base);
      finish(C, buf, total, base, false);
    }
  }
  if (pC >= 0) finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
  cand = warp_sum_ull(cand);
  if (lane == 0 && cand) { atomicAdd(&H->cand[LST_T3_], cand); atomicAdd(&H->eval[LST_T3_], cand); }
}

// ------------------------------------------------------------------------------------------
// a4: quintuplets.  Owner = inner triplet A = (m1, m2, m3); candidates are the triplets whose
// first MD is m3: [t3_start[seg_start[m3]], t3_start[seg_start[m3 + 1]]), contiguous because
// triplets are stored by first segment and segments by inner MD.  Two levels: the curvature match
// Q2 (one 4-byte load and a compare) on every candidate, survivors compacted into a queue; the
// two fits on full tiles of survivors.
// ------------------------------------------------------------------------------------------
constexpr int kT5Stash = 64;
struct T5Warp {
  float4 p[3][32];
  float kA[32];
  int layer[32], tab[32];
  int2 q[kQueue];
  int cnt[2][32];
  int stI[2][kT5Stash];
  float stV[2][3][kT5Stash];
};

__device__ __forceinline__ void t5_emit(const Params& P, const Slot& S, int pos, int A, int B, float kfit, float chi2xy,
                                        float chi2rz) {
  if (pos >= P.L.cap_t5) return;
  const int4 ta = S.t3_pack()[A], tb = S.t3_pack()[B];
  int* md = S.t5_md() + 5 * (size_t)pos;
  md[0] = ta.x; md[1] = ta.y; md[2] = ta.z; md[3] = tb.y; md[4] = tb.z;
  S.t5_t3()[pos] = make_int2(A, B);
  S.t5_score()[pos] = chi2xy + chi2rz;   // [D] D1, one fp32 addition of the fp32 values whatever the store
  S.t5_kfit()[pos] = kfit;               // [P] P1 reads the fitted curvature in fp32 whatever the store
  if (P.store_half) {   // [H]
    __half* f = reinterpret_cast<__half*>(S.t5_f()) + 5 * (size_t)pos;
    f[0] = __float2half_rn(__int_as_float(ta.w)); f[1] = __float2half_rn(__int_as_float(tb.w)); f[2] = __float2half_rn(kfit);
    f[3] = __float2half_rn(chi2xy); f[4] = __float2half_rn(chi2rz);
  } else {
    float* f = S.t5_f() + 5 * (size_t)pos;
    f[0] = __int_as_float(ta.w); f[1] = __int_as_float(tb.w); f[2] = kfit; f[3] = chi2xy; f[4] = chi2rz;
  }
}

template <bool DIRECT>
__device__ __forceinline__ int t5_walk(const Params& P, const Slot& S, T5Warp& sh, int buf, int n, int off, int total,
                                       int B0, int A0, int base) {
  const int4* t3_pack = S.t3_pack();
  const float4* anchor = S.md_anchor();
  const int lane = (int)lane_id();
  const float dk = P.cuts.t5_dkappa_max;
  int running = 0, qh = 0, qt = 0;
  auto fits = [&](bool valid, int2 it) {
    bool pass = false;
    T5Out o;
    const int ol = it.x, Bi = it.y;
    if (valid) {
      const int4 tb = t3_pack[Bi];
      const float4 p[5] = {sh.p[0][ol], sh.p[1][ol], sh.p[2][ol], anchor[tb.y], anchor[tb.z]};
      pass = t5_select(P.cuts, sh.layer[ol], sh.kA[ol], __int_as_float(tb.w), p, o);
    }
    const unsigned bal = __ballot_sync(kFull, pass);
    if (pass) {
      const int pos = running + __popc(bal & lanemask_lt());
      if (!DIRECT) {
        atomicAdd(&sh.cnt[buf][ol], 1);
        if (pos < kT5Stash) {
          sh.stI[buf][pos] = (ol << 26) | Bi;
          sh.stV[buf][0][pos] = o.kfit; sh.stV[buf][1][pos] = o.chi2xy; sh.stV[buf][2][pos] = o.chi2rz;
        }
      } else {
        t5_emit(P, S, base + pos, A0 + ol, Bi, o.kfit, o.chi2xy, o.chi2rz);
      }
    }
    running += __popc(bal);
  };
  auto drain = [&](bool all) {
    while (qt - qh >= 32 || (all && qt > qh)) {
      __syncwarp();
      const bool valid = lane < qt - qh;
      int2 it = make_int2(0, 0);
      if (valid) it = sh.q[(qh + lane) & (kQueue - 1)];
      fits(valid, it);
      qh += min(32, qt - qh);
      __syncwarp();
    }
  };
  for (int tb = 0; tb < total; tb += 32) {
    const int rk = tile_owner(n, off, tb);
    const int j = tb + lane;
    const int ol = (j < total) ? sh.tab[rk] : 0;
    const int Bi = __shfl_sync(kFull, B0, ol) + (j - __shfl_sync(kFull, off, ol));
    bool keep = false;
    if (j < total) keep = fabsf(sh.kA[ol] - __int_as_float(t3_pack[Bi].w)) <= dk;   // Q2, exactly as t5_select
    const unsigned bal = __ballot_sync(kFull, keep);
    if (keep) sh.q[(qt + __popc(bal & lanemask_lt())) & (kQueue - 1)] = make_int2(ol, Bi);
    qt += __popc(bal);
    drain(false);
  }
  drain(true);
  return running;
}

__global__ void __launch_bounds__(kWarps * 32, LST_T5_BLOCKS) k_t5(const __grid_constant__ Params P) {
  __shared__ T5Warp shw[kWarps];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int cap = P.L.cap_t5;
  const int nAll = H->n[LST_T3_];
  // only triplets starting on layer 0 or 1 can be the inner half of a quintuplet: a prefix of the triplet list when module ids
  // are ordered by layer (P.live_modules[0]); only they are walked, the CSR entries of the rest are filled in by the warp of
  // the last chunk
  int nT3 = nAll;
  if (P.live_modules[0] < P.L.n_modules && !H->overflow)
    nT3 = min(nAll, S.t3_start()[S.seg_start()[S.md_start()[P.live_modules[0]]]]);
  const int nChunks = (nT3 + kChunk - 1) / kChunk;
  const int lane = (int)lane_id();
  T5Warp& sh = shw[threadIdx.x >> 5];
  const int* seg_start = S.seg_start();
  const int* t3_start = S.t3_start();
  int* t5_start = S.t5_start();
  unsigned long long* status = S.lb(LST_T5_);
  unsigned long long cand = 0;

  auto finish = [&](int C, int b, int total, int base, bool from_stash) {
    const int A0 = C * kChunk, A = A0 + lane;
    if (from_stash)
      for (int t = lane; t < total; t += 32) {
        const int v = sh.stI[b][t];
        t5_emit(P, S, base + t, A0 + (int)((unsigned)v >> 26), v & (kMaxCap - 1), sh.stV[b][0][t], sh.stV[b][1][t],
                sh.stV[b][2][t]);
      }
    int tot;
    const int ex = warp_excl_scan(sh.cnt[b][lane], tot);
    if (A < nT3) t5_start[A] = min(base + ex, cap);
    if (A0 + 31 >= nT3 - 1) {
      fill_ints(t5_start, nT3, nAll + 1, min(base + total, cap));
      if (A == nT3 - 1) publish_total(H, LST_T5_, base + total, cap);
    }
    __syncwarp();
  };

  int buf = 0, pC = -1, pTotal = 0;
  for (;;) {
    const int C = warp_ticket(&H->ticket[LST_T5_]);
    if (C >= nChunks) {
      if (C == 0) {
        fill_ints(t5_start, 0, nAll + 1, 0);
        if (lane == 0) publish_total(H, LST_T5_, 0, cap);
      }
      break;
    }
    const int A0 = C * kChunk, A = A0 + lane;
    int n = 0, B0 = 0;
    if (A < nT3) {
      // every load of the owner's record is issued before any is needed: the chains travel together
      const int4 ta = S.t3_pack()[A];
      const int g0 = seg_start[ta.z], g1 = seg_start[ta.z + 1];
      const float4 q0 = S.md_anchor()[ta.x], q1 = S.md_anchor()[ta.y], q2 = S.md_anchor()[ta.z];
      const int layer = P.mod_layer[S.md_module()[ta.x]];
      B0 = t3_start[g0];
      n = t3_start[g1] - B0;
      sh.p[0][lane] = q0;
      sh.p[1][lane] = q1;
      sh.p[2][lane] = q2;
      sh.kA[lane] = __int_as_float(ta.w);
      sh.layer[lane] = layer;
      if (layer > 1) n = 0;   // cannot happen with a valid module map (targets one layer out); t5_select indexes [layer + 4]
    }
    sh.cnt[buf][lane] = 0;
    cand += (unsigned long long)n;
    int total_c;
    const int off = warp_excl_scan(n, total_c);
    build_owner_table(n, sh.tab);
    const int total = t5_walk<false>(P, S, sh, buf, n, off, total_c, B0, A0, 0);
    publish_aggregate(status, C, total);
    __syncwarp();
    if (pC >= 0) {
      finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
      pC = -1;
    }
    if (total <= kT5Stash) {
      pC = C; pTotal = total; buf ^= 1;
    } else {
      if (lane == 0) atomicAdd(&H->rewalk[LST_T5_], 1ull);
      const int base = resolve_base(status, C, total);
      t5_walk<true>(P, S, sh, buf, n, off, total_c, B0, A0, base);
      finish(C, buf, total, base, false);
    }
  }
  if (pC >= 0) finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
  cand = warp_sum_ull(cand);
  if (lane == 0 && cand) { atomicAdd(&H->cand[LST_T5_], cand); atomicAdd(&H->eval[LST_T5_], cand); }
}

// ------------------------------------------------------------------------------------------
// [D] duplicate cleaning of quintuplets (DESIGN.md section 1 [D]; optional stage LST_CLEAN).
// Two quintuplets that share >= 6 of their 10 original hits share a mini-doublet (a mini-doublet is a
// pair of hits of one module: without a common MD at most one hit per common layer can coincide, 5 in all;
// lst_create refuses t5_dup_min_shared < 6), so the
// partners of a quintuplet are found through an MD -> quintuplets incidence table (counting sort over the
// MDs: count, scan, fill), and every (quintuplet, partner) pair goes through the exact rule D2-D4.
// The result does not depend on the order of the incidence lists: D4 is an "exists" over the partners.
// ------------------------------------------------------------------------------------------
// hit tuple in layer order (the score was stored by the quintuplet kernel); zero the incidence counters
__global__ void __launch_bounds__(256) k_clean_prepare(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  const SlotHeader* H = S.hdr();
  const int n5 = H->n[LST_T5_], nmd = H->n[LST_MD_];
  int* cnt = S.inc_start();
  int* cur = S.inc_cur();
  const int2* mh = S.md_hits();
  const int nz = (nmd + 1 + 3) / 4 * 4;   // the in-place scan reads whole int4s
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < max(n5, nz); i += gridDim.x * blockDim.x) {
    if (i < nz) { cnt[i] = 0; cur[i] = 0; }
    if (i < n5) {
      S.t5_keep()[i] = 1;
      const int* md = S.t5_md() + 5 * (size_t)i;
      int2* out = reinterpret_cast<int2*>(S.t5_hits()) + 5 * (size_t)i;
#pragma unroll
      for (int k = 0; k < 5; ++k) out[k] = mh[md[k]];
    }
  }
}

// quintuplets per MD (k_scan turns the counts into offsets)
__global__ void __launch_bounds__(256) k_clean_count(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  const int n5 = S.hdr()->n[LST_T5_];
  int* cnt = S.inc_start();
  const int* md = S.t5_md();
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < 5 * n5; j += gridDim.x * blockDim.x) atomicAdd(cnt + md[j], 1);
}

__global__ void __launch_bounds__(256) k_clean_fill(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  const int n5 = S.hdr()->n[LST_T5_];
  const int* start = S.inc_start();
  int* cur = S.inc_cur();
  int2* list = S.inc_list();
  const int* md = S.t5_md();
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < 5 * n5; j += gridDim.x * blockDim.x) {
    const int m = md[j];
    list[start[m] + atomicAdd(cur + m, 1)] = make_int2(j / 5, m);
  }
}

// A hit belongs to one layer and one sensor side, so it can sit at one position only of a quintuplet's tuple:
// with OFF = (position of a common MD in q) - (its position in b), MD i of q can only equal MD i - OFF of b and
// hit k of q only hit k - 2 OFF of b.  Quintuplets span 5 of the 6 layers, so OFF is -1, 0 or 1.
template <int OFF>
__device__ __forceinline__ void common_mds(const int (&qm)[5], const int (&bm)[5], int pos, int& n_md, bool& earlier) {
  n_md = 0;
  earlier = false;
#pragma unroll
  for (int i = 0; i < 5; ++i) {
    if (i - OFF < 0 || i - OFF >= 5) continue;
    const bool eq = qm[i] == bm[i - OFF];
    n_md += eq;
    earlier = earlier || (eq && i < pos);
  }
}
template <int OFF>
__device__ __forceinline__ int common_hits(const int (&a)[10], const int (&h)[10]) {
  int shared = 0;
#pragma unroll
  for (int k = 0; k < 10; ++k)
    if (k - 2 * OFF >= 0 && k - 2 * OFF < 10) shared += (a[k] == h[k - 2 * OFF]);
  return shared;
}

// One thread per entry of the incidence table = (quintuplet q, one of its five MDs): rule D2-D4 against every
// quintuplet in that MD's list.  Threads are taken in TABLE order, so neighbouring threads walk the same list
// (same trip count, the partners' records served from L1).
// A removal is an idempotent store of 0 (k_clean_prepare set every flag to 1); k_clean_list then lists the kept ones.
__global__ void __launch_bounds__(256) k_clean_mark(const __grid_constant__ Params P) {
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int n5 = H->n[LST_T5_];
  const int* start = S.inc_start();
  const int2* list = S.inc_list();
  const int* md = S.t5_md();
  const int* hits = S.t5_hits();
  const float* score = S.t5_score();
  unsigned char* keep = S.t5_keep();
  const int K = P.dup_min_shared;
  for (int t = blockIdx.x * blockDim.x + threadIdx.x; t < 5 * n5; t += gridDim.x * blockDim.x) {
    const int2 entry = list[t];
    const int q = entry.x, m = entry.y;
    const int j0 = start[m], j1 = start[m + 1];
    if (j1 - j0 < 2) continue;                              // the list holds q itself only
    int qm[5];
#pragma unroll
    for (int k = 0; k < 5; ++k) qm[k] = md[5 * (size_t)q + k];
    int pos = 0;
#pragma unroll
    for (int k = 1; k < 5; ++k) pos = (qm[k] == m) ? k : pos;
    const float sq = score[q];
    bool removed = false;
    for (int j = j0; j < j1 && !removed; ++j) {
      const int b = list[j].x;
      if (b == q) continue;
      // common MDs first: a common MD is two common hits, and a layer without a common MD holds at most one
      // common hit, so  2 * n_md <= shared <= n_md + 5 : most pairs are decided without looking at the hits
      int bm[5];
#pragma unroll
      for (int k = 0; k < 5; ++k) bm[k] = md[5 * (size_t)b + k];
      int kpos = 0;
#pragma unroll
      for (int k = 1; k < 5; ++k) kpos = (bm[k] == m) ? k : kpos;
      const int off = pos - kpos;
      int n_md = 0;
      bool earlier = false;
      if (off == 0) common_mds<0>(qm, bm, pos, n_md, earlier);
      else if (off == 1) common_mds<1>(qm, bm, pos, n_md, earlier);
      else if (off == -1) common_mds<-1>(qm, bm, pos, n_md, earlier);
      else {   // not reachable with 6 layers; the position-free form
#pragma unroll
        for (int k = 0; k < 5; ++k)
#pragma unroll
          for (int i = 0; i < 5; ++i) {
            const bool eq = qm[i] == bm[k];
            n_md += eq;
            earlier = earlier || (eq && i < pos);
          }
      }
      if (earlier) continue;                                // the thread of the earlier common MD handles this pair
      bool dup = 2 * n_md >= K;
      const bool need_hits = !dup && n_md + 5 >= K;
      const float sb = score[b];
      if (!need_hits && (!dup || sb != sq)) {               // decided by the MDs and the scores alone
        removed = dup && sb < sq;
        continue;
      }
      int a[10], h[10];
#pragma unroll
      for (int k = 0; k < 10; ++k) { a[k] = hits[10 * (size_t)q + k]; h[k] = hits[10 * (size_t)b + k]; }
      if (need_hits) {
        int shared = 0;                                     // D2: the 10 hits of a quintuplet are distinct
        if (off == 0) shared = common_hits<0>(a, h);
        else if (off == 1) shared = common_hits<1>(a, h);
        else if (off == -1) shared = common_hits<-1>(a, h);
        else {
#pragma unroll
          for (int i = 0; i < 10; ++i)
#pragma unroll
            for (int k = 0; k < 10; ++k) shared += (a[i] == h[k]);
        }
        dup = shared >= K;
      }
      if (!dup) continue;
      bool beats = sb < sq;                                 // D3
      if (sb == sq) {
#pragma unroll
        for (int k = 9; k >= 0; --k)
          if (h[k] != a[k]) beats = h[k] < a[k];            // the first differing position decides
      }
      removed = beats;
    }
    if (removed) keep[q] = 0;
  }
}

// The kept quintuplets in ascending order (the T5-only track-candidate list): one block of 1024 threads per event,
// 8 flags per thread and step.
__global__ void __launch_bounds__(1024) k_clean_list(const __grid_constant__ Params P) {
  __shared__ int s_warp[32];
  __shared__ int s_base;
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int n5 = H->n[LST_T5_];
  const unsigned char* keep = S.t5_keep();
  int* tc = S.tc_list();
  const int w = threadIdx.x >> 5;
  if (threadIdx.x == 0) s_base = 0;
  __syncthreads();
  for (int q0 = 0; q0 < n5; q0 += 8192) {
    const int q = q0 + 8 * threadIdx.x;
    unsigned long long f = 0;
    if (q < n5) f = *reinterpret_cast<const unsigned long long*>(keep + q);   // the array is padded to 256 B
    if (q + 8 > n5) f &= (q < n5) ? ((1ull << (8 * (n5 - q))) - 1ull) : 0ull;
    const int mine = __popcll(f & 0x0101010101010101ull);
    const int incl = warp_incl_scan(mine);
    if (lane_id() == 31) s_warp[w] = incl;
    __syncthreads();
    int before = s_base, total = 0;
#pragma unroll 8
    for (int i = 0; i < 32; ++i) {
      before += (i < w) ? s_warp[i] : 0;
      total += s_warp[i];
    }
    int pos = before + incl - mine;
#pragma unroll
    for (int k = 0; k < 8; ++k)
      if ((f >> (8 * k)) & 1ull) tc[pos++] = q + k;
    __syncthreads();
    if (threadIdx.x == 0) s_base += total;
    __syncthreads();
  }
  if (threadIdx.x == 0) H->n_kept = s_base;
}

// ------------------------------------------------------------------------------------------
// [P] pixel line segments -> pixel triplets / pixel quintuplets (DESIGN.md section 1 [P]; optional
// stage LST_PIXEL).  The method's search space is the full product (outer object, seed); here the seeds are binned by the
// azimuth of their direction at the beam line, and an object looks only at the bins its first anchor allows:
// with phi_p the azimuth of the first anchor (x, y, r) and delta = phi0 - phi_p, the P2 term of that anchor is
//     e = (kappa / 2) r^2 + x sin phi0 - y cos phi0 = (kappa / 2) r^2 + n r sin(delta),   n = |(cos phi0, sin phi0)|,
// P2 needs e^2 / var_xy[layer] <= chi2xy_max (every term of the sum is >= 0), P1 confines kappa to kappa_obj +- dkappa_max
// and P0 confines delta to (-pi/2, pi/2): an interval of sin(delta), hence of phi0.  Every seed inside the window goes
// through the exact selection, so the link set does not depend on the window.  Seeds whose direction is not a unit vector
// (|n^2 - 1| > 1e-3) have no such window: they sit in a bin of their own that every object looks at.  The bins are
// (curvature band, azimuth): P1 is the second window (seed_band_of below).
// ------------------------------------------------------------------------------------------
constexpr float kPiF = 3.14159274f;
constexpr float kSeedBinScale = 81.4873309f;   // kSeedPhiBins / (2 pi)
// Curvature bands: band(kappa) = clamp(floor((kappa + 0.016) * 500), 0, kSeedBands - 1): width 0.002 per cm, the two edge bands
// open-ended; monotone in kappa.  A seed is filed under every band from band(kappa - dkw) to band(kappa + dkw), dkw = the larger
// pix_dkappa_max with slack, so the ONE band of an object's own curvature holds every seed P1 can accept for it.
constexpr float kBandOffset = 0.016f, kBandScale = 500.0f;
static_assert(kSeedPhiBins == 512 && kSeedBands == 16 && kSeedBins == 8192, "k_seed_bin scans eight bins per thread");

__device__ __forceinline__ int seed_band_of(float kappa) {
  return (int)fminf(fmaxf(floorf((kappa + kBandOffset) * kBandScale), 0.0f), (float)(kSeedBands - 1));
}
__device__ __forceinline__ float seed_band_reach(const Cuts& c) {
  const float d = fmaxf(c.pix_dkappa_max[0], c.pix_dkappa_max[1]) * 1.001f + 1e-7f;
  return d >= 0.0f ? d : 0.0f;
}
// kSeedBins + 1: no object can accept the seed (a non-finite direction makes e infinite or NaN, a zero direction fails P0, a NaN
// curvature fails P1); kSeedBins: direction not a unit vector; else the azimuth bin.
__device__ __forceinline__ int seed_phi_bin_of(float kappa, float c, float s) {
  if (!(fabsf(c) <= 3.4028235e38f) || !(fabsf(s) <= 3.4028235e38f) || (c == 0.0f && s == 0.0f) || kappa != kappa) return kSeedBins + 1;
  const float n2 = c * c + s * s;
  if (!(fabsf(n2 - 1.0f) <= 1e-3f)) return kSeedBins;
  const int b = (int)floorf((atan2f(s, c) + kPiF) * kSeedBinScale);
  return min(kSeedPhiBins - 1, max(0, b));
}

// One block per event: histogram over the (band, azimuth) bins in shared memory, scan, scatter of the records (kappa, cos, sin,
// z0), (t, original index) -- once per band the seed is filed under.  The order inside a bin is the arrival order (it never
// reaches the output: links carry the original seed index and are ordered by it).  Also clears the look-back words and the
// counters of the two link kernels.
__global__ void __launch_bounds__(1024) k_seed_bin(const __grid_constant__ Params P, const __grid_constant__ SeedBatch B) {
  __shared__ int s_cnt[kSeedBins + 2], s_warp[32];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const SeedInput& in = B.ev[blockIdx.y];
  const int n = min(in.n, P.L.cap_seeds);
  const int tid = (int)threadIdx.x, lane = (int)lane_id();
  const float reach = seed_band_reach(P.cuts);
  for (int i = tid; i < kSeedBins + 2; i += 1024) s_cnt[i] = 0;
  int4* lb = S.at<int4>(P.L.lb_pix[0]);
  for (int i = tid; i < (int)(P.L.lb_pix_bytes / 16); i += 1024) lb[i] = make_int4(0, 0, 0, 0);
  __syncthreads();
  for (int i = tid; i < n; i += 1024) {
    const float k = in.kappa[i];
    const int pb = seed_phi_bin_of(k, in.cphi[i], in.sphi[i]);
    if (pb >= kSeedBins) {
      atomicAdd(&s_cnt[pb], 1);
    } else {
      const int b1 = seed_band_of(k + reach);
      for (int b = seed_band_of(k - reach); b <= b1; ++b) atomicAdd(&s_cnt[b * kSeedPhiBins + pb], 1);
    }
  }
  __syncthreads();
  // exclusive scan of the kSeedBins counters, eight per thread; the counters become the scatter cursors
  int v[8], mine = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) { v[k] = s_cnt[8 * tid + k]; mine += v[k]; }
  const int incl = warp_incl_scan(mine);
  if (lane == 31) s_warp[tid >> 5] = incl;
  __syncthreads();
  if (tid < 32) {
    const int w = s_warp[tid];
    s_warp[tid] = warp_incl_scan(w) - w;
  }
  __syncthreads();
  int ex = s_warp[tid >> 5] + incl - mine;
  int* start = S.seed_bin_start();
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    s_cnt[8 * tid + k] = ex;
    start[8 * tid + k] = ex;
    ex += v[k];
  }
  if (tid == 1023) {
    const int n_wild = s_cnt[kSeedBins], n_dead = s_cnt[kSeedBins + 1];
    s_cnt[kSeedBins] = ex;
    s_cnt[kSeedBins + 1] = ex + n_wild;
    start[kSeedBins] = ex;
    start[kSeedBins + 1] = ex + n_wild;
    start[kSeedBins + 2] = ex + n_wild + n_dead;
  }
  __syncthreads();
  float4* rec4 = S.seed_rec4();
  float2* rec2 = S.seed_rec2();
  for (int i = tid; i < n; i += 1024) {
    const float k = in.kappa[i], c = in.cphi[i], sn = in.sphi[i];
    const float4 a = make_float4(k, c, sn, in.z0[i]);
    const float2 b2 = make_float2(in.t[i], __int_as_float(i));
    const int pb = seed_phi_bin_of(k, c, sn);
    if (pb >= kSeedBins) {
      const int pos = atomicAdd(&s_cnt[pb], 1);
      rec4[pos] = a;
      rec2[pos] = b2;
    } else {
      const int b1 = seed_band_of(k + reach);
      for (int b = seed_band_of(k - reach); b <= b1; ++b) {
        const int pos = atomicAdd(&s_cnt[b * kSeedPhiBins + pb], 1);
        rec4[pos] = a;
        rec2[pos] = b2;
      }
    }
  }
  if (tid == 0) {
    H->n_seeds = n;
    atomicAnd(&H->overflow, ~0x30);
    for (int k = 0; k < 2; ++k) {
      H->n_pix[k] = 0;
      H->ticket_pix[k] = 0u;
      H->needed_pix[k] = H->cand_pix[k] = H->eval_pix[k] = H->rewalk_pix[k] = 0ull;
    }
  }
}

constexpr int kPixWarps = 4;
constexpr int kPixStash = 64;
template <int N>
struct PixWarp {
  float4 p[N][32];
  float kobj[32];
  int layer[32], tab[32];
  int2 q[kQueue];
  int cnt[2][32];
  int stSeed[2][kPixStash], stOl[2][kPixStash];
  float stV[2][3][kPixStash];
};

template <int KIND>
__device__ __forceinline__ void pix_emit(const Params& P, const Slot& S, int pos, int obj, int seed, float chi2xy, float chi2rz,
                                         float dk) {
  if (pos >= P.L.cap_pix[KIND]) return;
  S.pix_link(KIND)[pos] = make_int2(seed, obj);
  float* f = S.pix_f(KIND) + 3 * (size_t)pos;
  f[0] = chi2xy; f[1] = chi2rz; f[2] = dk;
}

// Owner lane: `n` candidates = n1 binned seeds starting at position `first` of the bin-ordered seed list, then nMain - n1
// starting at `second` (the azimuth window may straddle +-pi: the tail and the head of the band), then all seeds of the
// non-unit bin, which starts at `wild0`.
// Two levels: P1, P0 and the first anchor's term of P2 on every candidate (one 16-byte load), survivors compacted
// into a queue; the full selection on full tiles of survivors.
template <int KIND, bool DIRECT>
__device__ __forceinline__ int pix_walk(const Params& P, const Slot& S, PixWarp<(KIND ? 5 : 3)>& sh, int buf, int n, int off,
                                        int total, int first, int n1, int second, int nMain, int wild0, int A0, int base) {
  constexpr int N = KIND ? 5 : 3;
  const float4* rec4 = S.seed_rec4();
  const float2* rec2 = S.seed_rec2();
  const int lane = (int)lane_id();
  const float dkmax = P.cuts.pix_dkappa_max[KIND], cxy = P.cuts.pix_chi2xy_max[KIND];
  int running = 0, qh = 0, qt = 0;
  auto full = [&](bool valid, int2 it) {
    bool pass = false;
    PixOut o;
    int orig = 0;
    const int ol = it.x;
    if (valid) {
      const float4 a = rec4[it.y];
      const float2 b = rec2[it.y];
      orig = __float_as_int(b.y);
      float4 p[N];
#pragma unroll
      for (int i = 0; i < N; ++i) p[i] = sh.p[i][ol];
      pass = pix_select<N>(P.cuts, KIND, sh.layer[ol], a.x, a.y, a.z, a.w, b.x, sh.kobj[ol], p, o);
    }
    const unsigned bal = __ballot_sync(kFull, pass);
    if (pass) {
      const int pos = running + __popc(bal & lanemask_lt());
      if (!DIRECT) {
        atomicAdd(&sh.cnt[buf][ol], 1);
        if (pos < kPixStash) {
          sh.stSeed[buf][pos] = orig; sh.stOl[buf][pos] = ol;
          sh.stV[buf][0][pos] = o.chi2xy; sh.stV[buf][1][pos] = o.chi2rz; sh.stV[buf][2][pos] = o.dk;
        }
      } else {
        pix_emit<KIND>(P, S, base + pos, A0 + ol, orig, o.chi2xy, o.chi2rz, o.dk);
      }
    }
    running += __popc(bal);
  };
  auto drain = [&](bool all) {
    while (qt - qh >= 32 || (all && qt > qh)) {
      __syncwarp();
      const bool valid = lane < qt - qh;
      int2 it = make_int2(0, 0);
      if (valid) it = sh.q[(qh + lane) & (kQueue - 1)];
      full(valid, it);
      qh += min(32, qt - qh);
      __syncwarp();
    }
  };
  for (int tb = 0; tb < total; tb += 32) {
    const int rk = tile_owner(n, off, tb);
    const int j = tb + lane;
    const int ol = (j < total) ? sh.tab[rk] : 0;
    const int jj = j - __shfl_sync(kFull, off, ol);
    const int f0 = __shfl_sync(kFull, first, ol), m1 = __shfl_sync(kFull, n1, ol);
    const int f1 = __shfl_sync(kFull, second, ol), nm = __shfl_sync(kFull, nMain, ol);
    const int idx = jj < m1 ? f0 + jj : jj < nm ? f1 + (jj - m1) : wild0 + (jj - nm);
    bool keep = false;
    if (j < total) {
      const float4 a = rec4[idx];                     // kappa, cos, sin, z0
      const float4 p0 = sh.p[0][ol];
      const float hk = 0.5f * a.x;
      const float e = (hk * (p0.w * p0.w) + p0.x * a.z) - p0.y * a.y;    // the i = 0 term of P2, exactly as pix_select
      keep = fabsf(sh.kobj[ol] - a.x) <= dkmax && p0.x * a.y + p0.y * a.z > 0.0f &&
             (e * e) * P.cuts.pix_inv_var_xy[sh.layer[ol]] <= cxy;
    }
    const unsigned bal = __ballot_sync(kFull, keep);
    if (keep) sh.q[(qt + __popc(bal & lanemask_lt())) & (kQueue - 1)] = make_int2(ol, idx);
    qt += __popc(bal);
    drain(false);
  }
  drain(true);
  return running;
}

template <int KIND>
__global__ void __launch_bounds__(kPixWarps * 32, 6) k_pix(const __grid_constant__ Params P) {
  constexpr int N = KIND ? 5 : 3;
  __shared__ PixWarp<N> shw[kPixWarps];
  __shared__ float s_E[2];
  Slot S(P, blockIdx.y);
  SlotHeader* H = S.hdr();
  const int cap = P.L.cap_pix[KIND];
  const int nAll = H->n[KIND ? LST_T5_ : LST_T3_];
  // Triplets are numbered by first segment, segments by inner MD, MDs by module: when the module ids are ordered by layer
  // (P.live_modules[0] = number of leading modules on layers 0 and 1) the triplets that can be linked are a prefix of the
  // triplet list, found through the CSR offsets; only they are walked (this stage has no later stage reading its CSR array
  // inside the kernel chain, so the entries of the rest are simply filled in by the warp of the last chunk: measured against
  // sending the empty chunks through the ordered output, 81 against 98 us per 16 events).
  int nObj = nAll;
  if (!KIND && P.live_modules[0] < P.L.n_modules && !H->overflow)
    nObj = min(nAll, S.t3_start()[S.seg_start()[S.md_start()[P.live_modules[0]]]]);
  const int nChunks = (nObj + kChunk - 1) / kChunk;
  const int nSeeds = H->n_seeds;
  const int lane = (int)lane_id();
  PixWarp<N>& sh = shw[threadIdx.x >> 5];
  const int* bs = S.seed_bin_start();
  const int wild0 = bs[kSeedBins], nWild = bs[kSeedBins + 1] - wild0;
  int* pix_start = S.pix_start(KIND);
  unsigned long long* status = S.lb_pix(KIND);
  unsigned long long cand = 0, evals = 0;
  // largest |e| the first anchor may have, by its layer, with slack far above the rounding of e
  if (threadIdx.x < 2) s_E[threadIdx.x] = sqrtf(P.cuts.pix_chi2xy_max[KIND] / P.cuts.pix_inv_var_xy[threadIdx.x]) * 1.0001f + 1e-4f;
  __syncthreads();

  auto publish = [&](int total) {
    H->needed_pix[KIND] = (unsigned long long)total;
    H->n_pix[KIND] = min(total, cap);
    if (total > cap) atomicOr(&H->overflow, 16 << KIND);
  };
  // the links of one object in ascending ORIGINAL seed index (the order of the method's loop over the seeds): an
  // object has one or two links, so an insertion sort by its owner lane
  auto finish = [&](int C, int b, int total, int base, bool from_stash) {
    const int A0 = C * kChunk, A = A0 + lane;
    const int mine = sh.cnt[b][lane];
    int tot;
    const int ex = warp_excl_scan(mine, tot);
    if (from_stash) {
      for (int i = ex + 1; i < ex + mine; ++i) {
        const int key = sh.stSeed[b][i];
        const float v0 = sh.stV[b][0][i], v1 = sh.stV[b][1][i], v2 = sh.stV[b][2][i];
        int j = i - 1;
        for (; j >= ex && sh.stSeed[b][j] > key; --j) {
          sh.stSeed[b][j + 1] = sh.stSeed[b][j];
          sh.stV[b][0][j + 1] = sh.stV[b][0][j]; sh.stV[b][1][j + 1] = sh.stV[b][1][j]; sh.stV[b][2][j + 1] = sh.stV[b][2][j];
        }
        sh.stSeed[b][j + 1] = key;
        sh.stV[b][0][j + 1] = v0; sh.stV[b][1][j + 1] = v1; sh.stV[b][2][j + 1] = v2;
      }
      __syncwarp();
      for (int t = lane; t < total; t += 32)
        pix_emit<KIND>(P, S, base + t, A0 + sh.stOl[b][t], sh.stSeed[b][t], sh.stV[b][0][t], sh.stV[b][1][t], sh.stV[b][2][t]);
    } else {
      __syncwarp();   // the direct walk's stores of the other lanes
      int2* link = S.pix_link(KIND);
      float* f = S.pix_f(KIND);
      const int lo = min(base + ex, cap), hi = min(base + ex + mine, cap);
      for (int i = lo + 1; i < hi; ++i) {
        const int2 key = link[i];
        const float v0 = f[3 * (size_t)i], v1 = f[3 * (size_t)i + 1], v2 = f[3 * (size_t)i + 2];
        int j = i - 1;
        for (; j >= lo && link[j].x > key.x; --j) {
          link[j + 1] = link[j];
          f[3 * (size_t)(j + 1)] = f[3 * (size_t)j]; f[3 * (size_t)(j + 1) + 1] = f[3 * (size_t)j + 1]; f[3 * (size_t)(j + 1) + 2] = f[3 * (size_t)j + 2];
        }
        link[j + 1] = key;
        f[3 * (size_t)(j + 1)] = v0; f[3 * (size_t)(j + 1) + 1] = v1; f[3 * (size_t)(j + 1) + 2] = v2;
      }
    }
    if (A < nObj) pix_start[A] = min(base + ex, cap);
    if (A0 + 31 >= nObj - 1) {      // the last chunk: the end of the CSR array, for the objects not walked too
      fill_ints(pix_start, nObj, nAll + 1, min(base + total, cap));
      if (A == nObj - 1) publish(base + total);
    }
    __syncwarp();
  };

  int buf = 0, pC = -1, pTotal = 0;
  for (;;) {
    const int C = warp_ticket(&H->ticket_pix[KIND]);
    if (C >= nChunks) {
      if (C == 0) {
        fill_ints(pix_start, 0, nAll + 1, 0);
        if (lane == 0) publish(0);
      }
      break;
    }
    const int A0 = C * kChunk, A = A0 + lane;
    int n = 0, first = 0, n1 = 0, second = 0, nMain = 0;
    if (A < nObj) {
      int md[N];
      float kobj;
      if (KIND) {
        const int* m5 = S.t5_md() + 5 * (size_t)A;
#pragma unroll
        for (int i = 0; i < N; ++i) md[i] = m5[i];
        kobj = S.t5_kfit()[A];
      } else {
        const int4 ta = S.t3_pack()[A];
        md[0] = ta.x; md[1] = ta.y; md[2] = ta.z;
        kobj = __int_as_float(ta.w);
      }
      float4 pa[N];          // the anchors are fetched while the layer is looked up (two dependent loads)
#pragma unroll
      for (int i = 0; i < N; ++i) pa[i] = S.md_anchor()[md[i]];
      const int layer = P.mod_layer[S.md_module()[md[0]]];
      if (layer <= 1) {     // the first anchor of a pixel-linked object sits on one of the two innermost layers
        const float4 p0 = pa[0];
#pragma unroll
        for (int i = 0; i < N; ++i) sh.p[i][lane] = pa[i];
        sh.kobj[lane] = kobj;
        sh.layer[lane] = layer;
        cand += (unsigned long long)nSeeds;
        const float E = s_E[layer], r = p0.w;
        bool whole = !(E < 1.0e30f);
        if (!whole) {
          const float dk = P.cuts.pix_dkappa_max[KIND] * 1.001f + 1e-7f;
          const float hlo = 0.5f * (kobj - dk), hhi = 0.5f * (kobj + dk);
          float a = -E / r - hhi * r, b = E / r - hlo * r;     // range of n sin(delta)
          a -= fabsf(a) * 2e-3f + 1e-5f;
          b += fabsf(b) * 2e-3f + 1e-5f;
          if (a <= b && a <= 1.0f && b >= -1.0f) {
            const float phip = atan2f(p0.y, p0.x);
            const float lo = phip + asinf(fmaxf(a, -1.0f)) - 1e-4f, hi = phip + asinf(fminf(b, 1.0f)) + 1e-4f;
            int blo = (int)floorf((lo + kPiF) * kSeedBinScale) - 1, bhi = (int)floorf((hi + kPiF) * kSeedBinScale) + 1;
            if (bhi - blo + 1 >= kSeedPhiBins) {
              whole = true;
            } else {
              const int* band = bs + seed_band_of(kobj) * kSeedPhiBins;
              blo = ((blo % kSeedPhiBins) + kSeedPhiBins) % kSeedPhiBins;
              bhi = ((bhi % kSeedPhiBins) + kSeedPhiBins) % kSeedPhiBins;
              first = band[blo];
              if (blo <= bhi) {
                n1 = nMain = band[bhi + 1] - first;
              } else {
                n1 = band[kSeedPhiBins] - first;
                second = band[0];
                nMain = n1 + (band[bhi + 1] - second);
              }
            }
          }
        }
        if (whole) {
          const int* band = bs + seed_band_of(kobj) * kSeedPhiBins;
          first = band[0];
          n1 = nMain = band[kSeedPhiBins] - first;
        }
        n = nMain + nWild;
      }
    }
    sh.cnt[buf][lane] = 0;
    evals += (unsigned long long)n;
    int total_c;
    const int off = warp_excl_scan(n, total_c);
    build_owner_table(n, sh.tab);
    const int total = pix_walk<KIND, false>(P, S, sh, buf, n, off, total_c, first, n1, second, nMain, wild0, A0, 0);
    publish_aggregate(status, C, total);
    __syncwarp();
    if (pC >= 0) {
      finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
      pC = -1;
    }
    if (total <= kPixStash) {
      pC = C; pTotal = total; buf ^= 1;
    } else {
      if (lane == 0) atomicAdd(&H->rewalk_pix[KIND], 1ull);
      const int base = resolve_base(status, C, total);
      pix_walk<KIND, true>(P, S, sh, buf, n, off, total_c, first, n1, second, nMain, wild0, A0, base);
      finish(C, buf, total, base, false);
    }
  }
  if (pC >= 0) finish(pC, buf ^ 1, pTotal, resolve_base(status, pC, pTotal), true);
  cand = warp_sum_ull(cand);
  evals = warp_sum_ull(evals);
  if (lane == 0 && cand) atomicAdd(&H->cand_pix[KIND], cand);
  if (lane == 0 && evals) atomicAdd(&H->eval_pix[KIND], evals);
}

// ------------------------------------------------------------------------------------------
// output helpers: original-hit-index tuples and float payloads, one thread per object
// ------------------------------------------------------------------------------------------
// blockIdx.y = slot of the batch; the object count comes from the slot header (clamped to capacity).
// Destination: the slot's scratch area (lst_fetch_batch copies it to the host from there).
__global__ void __launch_bounds__(256) k_gather_hits(const __grid_constant__ Params P, int kind) {
  Slot S(P, blockIdx.y);
  const int w = kind == LST_MD_ ? 1 : kind == LST_SEG_ ? 2 : kind == LST_T3_ ? 3 : 5;   // MDs per object
  const size_t m = (size_t)(kind == LST_CLEAN_ ? S.hdr()->n_kept : S.hdr()->n[kind]) * w;
  const int2* mh = S.md_hits();
  int2* out = reinterpret_cast<int2*>(S.scratch());
  // one thread per (object, MD): a warp writes 256 contiguous bytes whatever the class
  for (size_t j = (size_t)blockIdx.x * blockDim.x + threadIdx.x; j < m; j += (size_t)gridDim.x * blockDim.x) {
    int md;
    if (kind == LST_MD_) {
      md = (int)j;
    } else if (kind == LST_SEG_) {
      md = reinterpret_cast<const int*>(S.seg_md())[j];
    } else if (kind == LST_T3_) {
      const size_t i = j / 3;
      md = reinterpret_cast<const int*>(S.t3_pack())[4 * i + (j - 3 * i)];
    } else if (kind == LST_T5_) {
      md = S.t5_md()[j];
    } else {
      const size_t i = j / 5;
      md = S.t5_md()[5 * (size_t)S.tc_list()[i] + (j - 5 * i)];
    }
    out[j] = mh[md];
  }
}

// Float payload of object i of class `kind`, column c, in the order of lst_fetch_values, read from either store.
// HALF: the binary16 payload (bits); otherwise the fp32 value.  Columns that the selections need in fp32 (sinA, r, kappa of a
// triplet) are rounded on the way out in the binary16 case.
template <bool HALF>
__device__ __forceinline__ auto payload(const Slot& S, int kind, size_t i, int c) {
  if constexpr (HALF) {
    const __half* mo = reinterpret_cast<const __half*>(S.md_out());
    if (kind == LST_MD_) return c == 0 ? __float2half_rn(S.md_aux()[i].y) : c == 3 ? __float2half_rn(S.md_anchor()[i].w) : mo[2 * i + (c - 1)];
    if (kind == LST_SEG_) return reinterpret_cast<const __half*>(S.seg_f())[4 * i + c];
    if (kind == LST_T3_) return c == 0 ? __float2half_rn(__int_as_float(S.t3_pack()[i].w)) : reinterpret_cast<const __half*>(S.t3_chi2())[i];
    return reinterpret_cast<const __half*>(S.t5_f())[5 * i + c];
  } else {
    if (kind == LST_MD_) return c == 0 ? S.md_aux()[i].y : c == 3 ? S.md_anchor()[i].w : reinterpret_cast<const float*>(S.md_out())[2 * i + (c - 1)];
    if (kind == LST_SEG_) return reinterpret_cast<const float*>(S.seg_f())[4 * i + c];
    if (kind == LST_T3_) return c == 0 ? __int_as_float(S.t3_pack()[i].w) : S.t3_chi2()[i];
    return S.t5_f()[5 * i + c];
  }
}
// The whole payload table [n][w] of a slot to `out`, one element per thread and step (coalesced writes).
template <bool HALF, class T>
__device__ __forceinline__ void write_payload(const Slot& S, int kind, int n, T* out, size_t tid, size_t nth) {
  const int src_kind = kind == LST_CLEAN_ ? LST_T5_ : kind;
  const int w = src_kind == LST_T3_ ? 2 : src_kind == LST_T5_ ? 5 : 4;
  const size_t m = (size_t)n * w;
  for (size_t j = tid; j < m; j += nth) {
    const size_t i = j / w;
    const int c = (int)(j - i * w);
    out[j] = payload<HALF>(S, src_kind, kind == LST_CLEAN_ ? (size_t)S.tc_list()[i] : i, c);
  }
}

// Float payload of a class in the layout of lst_fetch_values to the slot's scratch area (pageable destination buffers).
__global__ void __launch_bounds__(256) k_pack_values(const __grid_constant__ Params P, int kind) {
  Slot S(P, blockIdx.y);
  const int n = kind == LST_CLEAN_ ? S.hdr()->n_kept : S.hdr()->n[kind];
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  if (P.store_half) write_payload<true>(S, kind, n, reinterpret_cast<__half*>(S.scratch()), tid, nth);
  else write_payload<false>(S, kind, n, reinterpret_cast<float*>(S.scratch()), tid, nth);
}

// Both tables of every slot of a batch straight into pinned (mapped) host buffers: the kernel IS the device-to-host
// copy -- each byte crosses PCIe once, in coalesced 128 / 256-byte writes -- and replaces two copy-engine calls per
// slot by ONE launch per batch.  Small grid: the kernel is bound by the link, not by the SMs.
__global__ void __launch_bounds__(256) k_fetch_direct(const __grid_constant__ Params P, const __grid_constant__ OutTable T, int kind) {
  Slot S(P, blockIdx.y);
  const int n = kind == LST_CLEAN_ ? S.hdr()->n_kept : S.hdr()->n[kind];   // LST_CLEAN_: the kept quintuplets only
  const size_t tid = (size_t)blockIdx.x * blockDim.x + threadIdx.x, nth = (size_t)gridDim.x * blockDim.x;
  if (int2* out = reinterpret_cast<int2*>(T.idx[blockIdx.y])) {
    const int w = kind == LST_MD_ ? 1 : kind == LST_SEG_ ? 2 : kind == LST_T3_ ? 3 : 5;
    const size_t m = (size_t)n * w;
    const int2* mh = S.md_hits();
    for (size_t j = tid; j < m; j += nth) {
      int md;
      if (kind == LST_MD_) md = (int)j;
      else if (kind == LST_SEG_) md = reinterpret_cast<const int*>(S.seg_md())[j];
      else if (kind == LST_T3_) { const size_t i = j / 3; md = reinterpret_cast<const int*>(S.t3_pack())[4 * i + (j - 3 * i)]; }
      else if (kind == LST_T5_) md = S.t5_md()[j];
      else { const size_t i = j / 5; md = S.t5_md()[5 * (size_t)S.tc_list()[i] + (j - 5 * i)]; }
      out[j] = mh[md];
    }
  }
  if (void* out = T.val[blockIdx.y]) {
    if (P.store_half) write_payload<true>(S, kind, n, reinterpret_cast<__half*>(out), tid, nth);
    else write_payload<false>(S, kind, n, reinterpret_cast<float*>(out), tid, nth);
  }
}

// ------------------------------------------------------------------------------------------
// launchers
// ------------------------------------------------------------------------------------------
#define LST_EV(k) do { if (ev) cudaEventRecord(ev[k], s); } while (0)

// blocks per event of a grid-stride / persistent kernel: enough to fill the machine across the batch
// The stage kernels are sized for HALF of what the machine holds: the kernels of two streams then run side by
// side, each event gets fewer warps (a stage's throughput per event stops growing long before a 16-event batch
// fills 148 SMs: ticket order and the ordered output bound it) and one stream's tail is filled by the other's body
// (measured: 44.0k -> 47.4k events/s on the 4 x 16 workload; a third or a quarter is no better).
constexpr int kGridShare = 2;
// Blocks per SM the grids are sized for (before the halving), from same-box sweeps in the 4-stream configuration; not the
// launch bounds (those set the register budget).  Segment kernel 4 / 5 / 6 / 7 / 8: 46.0 / 50.0 / 51.2 / 47.8 / 49.0 k events/s;
// the others are flat within 1 % (MD 5, T3 5, T5 6 together: 51.2 -> 51.6 k).
constexpr int kMdGrid = 5, kSegGrid = 6, kT3Grid = 5, kT5Grid = 6;
// lst_config.launches_in_flight >= 4 (Params::four_launches): the caller runs FOUR launches side by side, and the four streams do
// best in the same stage at the same time (profiles/r2_summary.md).  What counts is then whether the four launches of a stage
// TOGETHER fill a whole number of residency waves: waves x (148 SMs x resident blocks per SM) / (4 launches x events per launch).
//   k_seg  7 resident blocks per SM (1 036 slots), ONE wave: 16 blocks per event of a 16-event launch, 4 x 256 = 1 024 blocks
//   k_md, k_t3  6 per SM (888 slots), two waves: 27 per event, 4 x 432 = 1 728 <= 1 776;  k_t5 4 per SM, three waves: 27 per event
// Same-box sweep of the blocks per event (events/s, 4 x 16 events): k_seg 12 / 14 / 15 / 16 | 24 / 26 / 27 / 28 / 29 / 32 = 57.8 / 60.6 /
// 61.6 / 62.2 | 60.6 / 61.4 / 61.9 / 61.9 / 60.0 / 57.9 k (17 and 29 spill into a partial wave); with k_seg at 16, k_md + k_t3
// 13 / 23 / 27 / 41 = 61.7 / 62.1 / 62.5 / 61.4 k.  Alone such a k_seg launch takes 0.29 ms instead of 0.19: hence a hint, not the default.
constexpr int kMdGrid4 = 6, kSegGrid4 = 7, kT3Grid4 = 6, kSegShare4 = 4;
static int blocks_per_event(int wanted, int n_batch, int resident_per_sm, int share = 1) {
  const int per_event = max(8, 148 * resident_per_sm / (n_batch * share));
  return max(1, min(wanted, per_event));
}

int launch_bin(const Params& P, const HitBatch& src, int n_batch, cudaStream_t s, cudaEvent_t* ev, const StageIn* stage) {
  int n_max = 0;
  for (int b = 0; b < n_batch; ++b) n_max = max(n_max, src.ev[b].n);
  const unsigned nb = (unsigned)n_batch;
  // one hit per thread: the loads, the atomics and the scattered stores of all hits are in flight at once
  const dim3 g(max(1, (n_max + 255) / 256), nb);
  LST_EV(0);
  if (stage) {
    // Reading pinned host memory the kernel is PCIe bound (~75 KB in flight cover latency x bandwidth): a small
    // grid, on the library's own high-priority stream so that its blocks are placed ahead of the other streams'
    // stage kernels, and so that the stage-ins of all streams run one after the other at full link speed.
    cudaEventRecord(stage->before, s);
    cudaStreamWaitEvent(stage->stream, stage->before, 0);
    k_bin_count<<<dim3(min((int)g.x, 8), nb), 256, 0, stage->stream>>>(P, src);
    cudaEventRecord(stage->after, stage->stream);
    cudaStreamWaitEvent(s, stage->after, 0);
  } else {
    // grid-stride with about one wave of blocks: a block ends with a release fence (last_block_done) that waits for
    // its stores and atomics, so fewer, longer-lived blocks beat one hit per thread
    k_bin_count<<<dim3(blocks_per_event((int)g.x, n_batch, 8), nb), 256, 0, s>>>(P, src);
  }
  LST_EV(1);
  k_bin_scatter<<<g, 256, 0, s>>>(P, src);
  LST_EV(2);
  k_bin_order<<<dim3((max(n_max, P.L.n_modules) + 255) / 256, nb), 256, 0, s>>>(P);
  LST_EV(3);
  return 3;
}

int launch_stage(const Params& P, int n_batch, int stage, cudaStream_t s, cudaEvent_t* ev) {
  const unsigned nb = (unsigned)n_batch;
  LST_EV(0);
  switch (stage) {
    case LST_MD_:
      k_md<<<dim3(blocks_per_event((P.L.n_chunk[0] + kWarps - 1) / kWarps, n_batch, P.four_launches ? kMdGrid4 : kMdGrid, kGridShare), nb), kWarps * 32, 0, s>>>(P);
      break;
    case LST_SEG_:
      // (a module-owner walk with a flat on-chip key-window compare was built and measured in round 2: it lost, profiles/r2_seg_ab.md)
      k_seg<<<dim3(blocks_per_event((P.L.n_chunk[1] + kSegWarps - 1) / kSegWarps, n_batch, P.four_launches ? kSegGrid4 : kSegGrid, P.four_launches ? kSegShare4 : kGridShare), nb), kSegWarps * 32, 0, s>>>(P);
      break;
    case LST_T3_:
      k_t3<<<dim3(blocks_per_event((P.L.n_chunk[2] + kWarps - 1) / kWarps, n_batch, P.four_launches ? kT3Grid4 : kT3Grid, kGridShare), nb), kWarps * 32, 0, s>>>(P);
      break;
    case LST_T5_:
      k_t5<<<dim3(blocks_per_event((P.L.n_chunk[3] + kWarps - 1) / kWarps, n_batch, kT5Grid, kGridShare), nb), kWarps * 32, 0, s>>>(P);
      break;
    default:
      return 0;
  }
  LST_EV(1);
  return 1;
}

int launch_clean(const Params& P, int n_batch, cudaStream_t s, cudaEvent_t* ev) {
  const dim3 g(blocks_per_event((P.L.cap_t5 + 255) / 256, n_batch, 4), (unsigned)n_batch);
  LST_EV(0);
  k_clean_prepare<<<g, 256, 0, s>>>(P);
  LST_EV(1);
  k_clean_count<<<g, 256, 0, s>>>(P);
  k_scan<<<dim3(1, (unsigned)n_batch), 1024, 0, s>>>(P);
  LST_EV(2);
  k_clean_fill<<<g, 256, 0, s>>>(P);
  LST_EV(3);
  k_clean_mark<<<dim3(blocks_per_event((5 * P.L.cap_t5 + 255) / 256, n_batch, 8), (unsigned)n_batch), 256, 0, s>>>(P);
  k_clean_list<<<dim3(1, (unsigned)n_batch), 1024, 0, s>>>(P);
  LST_EV(4);
  return 6;
}

int launch_seed_bin(const Params& P, const SeedBatch& src, int n_batch, cudaStream_t s, cudaEvent_t* ev) {
  LST_EV(0);
  k_seed_bin<<<dim3(1, (unsigned)n_batch), 1024, 0, s>>>(P, src);
  LST_EV(1);
  return 1;
}

int launch_pixel(const Params& P, int n_batch, cudaStream_t s, cudaEvent_t* ev) {
  const unsigned nb = (unsigned)n_batch;
  LST_EV(0);
  k_pix<0><<<dim3(blocks_per_event((P.L.n_chunk_pix[0] + kPixWarps - 1) / kPixWarps, n_batch, 6, kGridShare), nb), kPixWarps * 32, 0, s>>>(P);
  LST_EV(1);
  k_pix<1><<<dim3(blocks_per_event((P.L.n_chunk_pix[1] + kPixWarps - 1) / kPixWarps, n_batch, 6, kGridShare), nb), kPixWarps * 32, 0, s>>>(P);
  LST_EV(2);
  return 2;
}

int launch_fetch_direct(const Params& P, const OutTable& T, int kind, int n_batch, cudaStream_t s) {
  k_fetch_direct<<<dim3(8, (unsigned)n_batch), 256, 0, s>>>(P, T, kind);
  return 1;
}

int launch_gather_hits(const Params& P, int kind, int n_max, int n_batch, cudaStream_t s) {
  if (n_max <= 0 || n_batch <= 0) return 0;
  const int w = kind == LST_MD_ ? 1 : kind == LST_SEG_ ? 2 : kind == LST_T3_ ? 3 : 5;
  k_gather_hits<<<dim3(min(256, (n_max * w + 255) / 256), (unsigned)n_batch), 256, 0, s>>>(P, kind);
  return 1;
}

int launch_pack_values(const Params& P, int kind, int n_max, int n_batch, cudaStream_t s) {
  if (n_max <= 0 || n_batch <= 0) return 0;
  k_pack_values<<<dim3(min(256, (n_max + 255) / 256), (unsigned)n_batch), 256, 0, s>>>(P, kind);
  return 1;
}

}  // namespace lst
