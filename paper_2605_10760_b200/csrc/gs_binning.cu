// gs_binning.cu -- steps a2-a5: per-tile instance lists ordered by (depth key, Gaussian index).
//
// Design (evidence: profiles/r1_v1_baseline.md -- a 6-pass one-sweep LSD radix sort of 64-bit (tile << 32 | depth)
// keys plus a serial per-thread duplication cost 112 + 40 us of a 614 us iteration): the sort on (tile, depth, index)
// keys is split MSD-first.
//   1. gs_preprocess counts the instances of every tile (atomics on tile_count) while it computes the rects.
//   2. tile_scan_kernel (multi-CTA, single pass, cooperative launch): exclusive prefix sum over the tile counts = the
//      per-tile ranges (step a5 comes for free), the instance total / overflow flag, and the tile order by descending
//      list-length class.
//   3. emit_kernel: every visible Gaussian appends (depth bits << 32 | index << 8 | region mask) to the bucket of each
//      tile of its rect (atomic cursor per tile) -- a counting-sort pass on the tile digit; the order inside a bucket is
//      arbitrary at this point.
//   4. tile_sort_kernel / tile_sort_large_kernel: every bucket is sorted on its 64-bit keys by a register-resident
//      bitonic network.  The keys are unique (the index is part of the key), so the result is THE (tile, depth bits,
//      index) order, bit for bit, whatever the arrival order was.  Buckets beyond 8192 keys are sorted in global memory.
// Integer work only.  Bytes: 8 I (emit) + 8 I (sort read) + 12 I (sorted keys + list entries) vs (8 + 24 * 6) I before.
#include <algorithm>

#include "gs_internal.cuh"
#include "gs_raster.cuh"

namespace gs {

constexpr int kSmallSortMax = 255;  // buckets up to this size are sorted by one warp (whole length/8 classes of the tile order)
constexpr int kMidSortMax = 2047;   // buckets up to this size are sorted by one CTA of 4 warps; beyond: the large kernel
constexpr int kLargeSort = 8192;    // up to this size: 512-thread CTA, 64 KB dynamic shared memory; beyond: global memory
// tile_count / tile_cursor are strided by 32 words (kCtrStride): one counter per 128-byte line, so that the atomics of
// different tiles are served by different L2 lines (3225 adjacent counters would share ~100 lines and serialise there)

// ---------------------------------------------------------------------------------------------------------------
// a2 + a5: prefix sum over the tile counts, ranges, totals, overflow flag, LPT tile order.
// ---------------------------------------------------------------------------------------------------------------
// Multi-CTA single-pass scan.  (Measured with clock64 on the one-CTA versions: ~20 k cycles whatever the algorithm --
// shared-memory atomics, L2 atomics or none -- because the 3225 strided counter loads and the ~3 x 3225 scattered
// stores of ONE SM retire about one sector per cycle.)  CTA b owns the tiles [b * TPC, (b + 1) * TPC), IT consecutive
// tiles per thread.  The block scan carries 9 words per thread: the instance count and 16 length-class counters packed
// as 16-bit fields, so one scan yields the per-tile ranges AND a stable counting sort of the tiles by length class
// (= the tile order); no atomics.  Every CTA publishes its 17 unpacked totals with an epoch flag and reads those of
// all the others (at most 128 CTAs; the launch is COOPERATIVE, so the runtime guarantees they are all co-resident and a
// CTA spinning on a sibling's flag cannot starve it), i.e. one L2 round trip instead of a second kernel.
constexpr int kScanT = 256;      // threads per CTA
constexpr int kScanWords = 9;    // [0] instances, [1..8] 16 class counters, two per word
constexpr int kScanCls = 16;
constexpr int kScanAgg = 1 + kScanCls;
constexpr int kScanMaxCta = 128;

// length class, longest first: 0: >= 2048, then half-octave steps 1536, 1024, 768, 512, ..., 24, 16; 15: < 16.
// Class 0 holds exactly the tiles beyond kMidSortMax, classes 0..6 those beyond kSmallSortMax.
__device__ __forceinline__ int length_class(uint32_t c) {
  if (c < 16u) return 15;
  const int e = 31 - __clz((int)c);
  const int q = 2 * e + (int)((c >> (e - 1)) & 1u);
  return max(22 - q, 0);
}

struct ScanVec { uint32_t w[kScanWords]; };

__device__ __forceinline__ ScanVec block_excl_scan_vec(const ScanVec& v, uint32_t (*wsum)[kScanWords], int lane, int warp,
                                                       ScanVec& total) {
  constexpr int NW = kScanT / 32;
  ScanVec incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
#pragma unroll
    for (int k = 0; k < kScanWords; ++k) {
      const uint32_t u = __shfl_up_sync(0xffffffffu, incl.w[k], d);
      if (lane >= d) incl.w[k] += u;
    }
  }
  if (lane == 31) {
#pragma unroll
    for (int k = 0; k < kScanWords; ++k) wsum[warp][k] = incl.w[k];
  }
  __syncthreads();
  ScanVec r;
#pragma unroll
  for (int k = 0; k < kScanWords; ++k) {
    uint32_t before = 0, all = 0;
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const uint32_t x = wsum[w][k];
      before += (w < warp) ? x : 0u;
      all += x;
    }
    r.w[k] = before + incl.w[k] - v.w[k];
    total.w[k] = all;
  }
  return r;
}

template <int IT>
__global__ void __launch_bounds__(kScanT)
tile_scan_kernel(int tiles, uint32_t* __restrict__ tile_count, uint32_t* __restrict__ tile_cursor,
                 uint2* __restrict__ ranges, uint32_t* __restrict__ order, uint32_t* agg, uint32_t* flags,
                 uint32_t epoch, int64_t capacity, Counts* counts, Counts* mailbox, uint32_t seq, Counts* counts_next) {
  __shared__ uint32_t wsum[kScanT / 32][kScanWords];
  __shared__ uint32_t s_pre[kScanAgg], s_tot[kScanAgg], s_base[kScanCls];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int b = blockIdx.x, nb = gridDim.x;
  const int t0 = (b * kScanT + tid) * IT;
  pdl_enter();
  if (tid < kScanAgg) { s_pre[tid] = 0; s_tot[tid] = 0; }
  uint32_t c[IT];
  int cls[IT];
  ScanVec v, total;
#pragma unroll
  for (int k = 0; k < kScanWords; ++k) v.w[k] = 0;
#pragma unroll
  for (int u = 0; u < IT; ++u) c[u] = (t0 + u < tiles) ? tile_count[(size_t)(t0 + u) * kCtrStride] : 0u;
  // counts_next != null: leave the counters this scan consumed, and the Counts record of the next iteration, zero
  if (counts_next) {
#pragma unroll
    for (int u = 0; u < IT; ++u)
      if (t0 + u < tiles) tile_count[(size_t)(t0 + u) * kCtrStride] = 0u;
    if (b == 0 && tid == 0) counts_next->n_visible = 0u;
  }
#pragma unroll
  for (int u = 0; u < IT; ++u) {
    cls[u] = length_class(c[u]);
    if (t0 + u < tiles) {
      v.w[0] += c[u];
#pragma unroll
      for (int w = 0; w < 8; ++w) v.w[1 + w] += ((cls[u] >> 1) == w) ? (1u << ((cls[u] & 1) * 16)) : 0u;
    }
  }
  ScanVec pref = block_excl_scan_vec(v, wsum, lane, warp, total);
  // publish this CTA's totals, then gather everybody's.  Every total travels as ONE 64-bit word {epoch, value}: the reader
  // spins on the word itself, so neither a flag nor a fence is needed (two L2 round trips less than flag-after-data)
  unsigned long long* agg64 = reinterpret_cast<unsigned long long*>(agg);
  if (tid < kScanAgg) {
    const uint32_t x = tid == 0 ? total.w[0] : (total.w[1 + ((tid - 1) >> 1)] >> (((tid - 1) & 1) * 16)) & 0xffffu;
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(agg64 + b * kScanAgg + tid), "l"(((unsigned long long)epoch << 32) | x) : "memory");
  }
  const uint32_t nvis = counts->n_visible;  // for the mailbox (off the critical path)
  for (int i = tid; i < nb * kScanAgg; i += kScanT) {
    const int j = i / kScanAgg, k = i - j * kScanAgg;
    unsigned long long w;
    // one 64-bit load per poll, in asm: left to the compiler (__ldcg) the word was split into a hoisted load of the value
    // half and a polled load of the epoch half -- stale totals whenever the scene changed
    do {
      asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(agg64 + i) : "memory");
    } while ((uint32_t)(w >> 32) != epoch);
    const uint32_t x = (uint32_t)w;
    if (x) {
      atomicAdd(&s_tot[k], x);
      if (j < b) atomicAdd(&s_pre[k], x);
    }
  }
  __syncthreads();
  const uint32_t I = s_tot[0];
  const bool ovf = (int64_t)I > capacity;
  if (tid == 0) {
    uint32_t bb = 0, nl = 0, nm = 0;
    for (int k = 0; k < kScanCls; ++k) {
      s_base[k] = bb + s_pre[1 + k];
      bb += s_tot[1 + k];
      if (k == 0) nl = bb;
      if (k == 6) nm = bb;
    }
    if (b == 0) {
      counts->n_instances = I;
      counts->overflow = ovf ? 1u : 0u;
      counts->n_large = nl;
      counts->n_mid = nm;
      counts->seq = seq;
      // one 16-byte store to the mapped host mailbox {n_visible, n_instances, overflow, seq}: a single posted write,
      // so no system-scope fence is needed to order the fields
      *reinterpret_cast<uint4*>(mailbox) = make_uint4(nvis, I, ovf ? 1u : 0u, seq);
      mailbox->n_large = nl;  // a hint for the next launch_binning (is the block-wide sort kernel needed at all?)
    }
  }
  __syncthreads();
  uint32_t off = s_pre[0] + pref.w[0];
#pragma unroll
  for (int u = 0; u < IT; ++u) {
    if (t0 + u < tiles) {
      tile_cursor[(size_t)(t0 + u) * kCtrStride] = off;
      // an iteration that overflows the instance capacity renders nothing
      ranges[t0 + u] = (c[u] && !ovf) ? make_uint2(off, off + c[u]) : make_uint2(0u, 0u);
      off += c[u];
      // tile ids by descending length class: class base + tiles of the class in earlier CTAs / threads / own tiles
      const int k = cls[u];
      uint32_t word = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) {
        const bool hit = (k >> 1) == w;
        word = hit ? pref.w[1 + w] : word;
        pref.w[1 + w] += hit ? (1u << ((k & 1) * 16)) : 0u;
      }
      order[s_base[k] + ((word >> ((k & 1) * 16)) & 0xffffu)] = (uint32_t)(t0 + u);
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// a3: duplication.  One thread per Gaussian; (depth bits << 32 | index) goes to the bucket of every tile of the rect.
// ---------------------------------------------------------------------------------------------------------------
constexpr int kEmitG = 32;    // visible Gaussians per CTA
constexpr int kEmitT = 128;   // threads per CTA

__global__ void __launch_bounds__(kEmitT)
emit_kernel(const uint4* __restrict__ vis_rec, const float4* __restrict__ feat, int tiles_x,
            uint32_t* __restrict__ tile_cursor, const Counts* __restrict__ counts, uint64_t* __restrict__ keys,
            bool exact_cull) {
  // Block-cooperative: the instances of the CTA's 32 Gaussians form one work list (prefix sum of the per-Gaussian tile
  // counts); every round the 128 threads take consecutive work items, whatever Gaussian they belong to, so a Gaussian
  // covering hundreds of tiles is emitted by the whole CTA; four independent atomics per thread are put in flight
  // before their results are used.  Small CTAs (many of them, few Gaussians each): the kernel is a chain of dependent
  // round trips (record -> cursor atomic -> key store), so what matters is how many chains are in flight per SM.
  // key = depth bits << 32 | index << 8 | region mask (the mask is a function of (index, tile): the order is unchanged)
  __shared__ uint32_t s_excl[kEmitG + 1], s_w[kEmitG], s_xy[kEmitG];
  __shared__ uint64_t s_key[kEmitG];
  __shared__ float4 s_f0[kEmitG];
  __shared__ MaskSetup s_ms[kEmitG];
  const int tid = threadIdx.x;
  pdl_enter();
  const uint32_t V = counts->n_visible;
  if (counts->overflow) return;
  // grid-stride over groups of 32 visible Gaussians: the host sizes the grid from the visible count of the last finished
  // iteration (two thirds of the N / 32 CTAs a worst-case grid needs would find nothing to do)
  for (uint32_t k0 = blockIdx.x * kEmitG; k0 < V; k0 += gridDim.x * kEmitG) {
  if (tid < 32) {
    const uint32_t k = k0 + tid;
    uint4 rec = make_uint4(0u, 0u, 0u, 0u);
    if (k < V) {
      rec = __ldg(vis_rec + k);
      s_f0[tid] = __ldg(feat + 3 * (size_t)k);  // the feature records are stored by visible slot
      const float4 f1 = __ldg(feat + 3 * (size_t)k + 1);
      s_ms[tid] = region_mask_setup(f1.x, f1.y, f1.z, f1.w);
    }
    const uint32_t w = (rec.y & 0xffffu) - (rec.x & 0xffffu), h = (rec.y >> 16) - (rec.x >> 16);
    const uint32_t n = w * h;
    uint32_t incl = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
      if (tid >= d) incl += v;
    }
    s_excl[tid] = incl - n;
    s_w[tid] = max(w, 1u);
    s_xy[tid] = rec.x;
    s_key[tid] = ((uint64_t)rec.z << 32) | ((uint64_t)rec.w << 8);
    if (tid == 31) s_excl[32] = incl;
  }
  __syncthreads();
  const uint32_t total = s_excl[kEmitG];
  for (uint32_t base = 0; base < total; base += kEmitT * 4) {
    uint32_t* cur[4];
    uint64_t kk[4];
    uint32_t pos[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t item = base + u * kEmitT + tid;
      cur[u] = nullptr;
      if (item < total) {
        int owner = 0;  // last Gaussian of the CTA whose exclusive prefix is <= item
#pragma unroll
        for (int step = kEmitG / 2; step >= 1; step >>= 1)
          if (s_excl[owner + step] <= item) owner += step;
        const uint32_t local = item - s_excl[owner], w = s_w[owner], xy = s_xy[owner];
        const uint32_t ty = (xy >> 16) + local / w, tx = (xy & 0xffffu) + local % w;
        cur[u] = &tile_cursor[(size_t)(ty * tiles_x + tx) * kCtrStride];
        // 8-bit mask of the tile's 8x4-pixel regions the ellipse {alpha >= 1/255} can reach (gs_raster.cuh), decided
        // ONCE per instance here instead of per (region, batch) in both compositing kernels
        const float4 f0 = s_f0[owner];
        const int pk = __float_as_int(f0.z);
        const float mx = (float)(((pk << 16) >> 16) - (int)tx * GS_TILE) + f0.x;
        const float my = (float)((pk >> 16) - (int)ty * GS_TILE) + f0.y;
        const uint32_t mask = region_mask(s_ms[owner], mx, my);
        kk[u] = s_key[owner] | (uint64_t)mask;
        // GS_OPT_EXACT_TILE_CULL: a tile of the rect that the ellipse itself does not reach (empty region mask) gets no
        // list entry at all; range_fix_kernel then shortens the tile's range to what was emitted
        if (exact_cull && mask == 0u) cur[u] = nullptr;
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) pos[u] = cur[u] ? atomicAdd(cur[u], 1u) : 0u;
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (cur[u]) keys[pos[u]] = kk[u];
  }
  __syncthreads();  // the shared records are rewritten by the next group
  }
}

// exact-cull mode only: the tile ranges were sized by the rect-based counts; shrink them to the emitted entries
__global__ void __launch_bounds__(256)
range_fix_kernel(int tiles, const uint32_t* __restrict__ tile_cursor, uint2* __restrict__ ranges) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  pdl_enter();
  if (t >= tiles) return;
  uint2 r = ranges[t];
  if (r.y > r.x) { r.y = min(r.y, tile_cursor[(size_t)t * kCtrStride]); if (r.y == r.x) r = make_uint2(0u, 0u); ranges[t] = r; }
}

// ---------------------------------------------------------------------------------------------------------------
// a4: per-bucket sort of the unique 64-bit keys; writes the sorted Gaussian ids.
// Normalised bitonic network: every comparator is ascending (first stage of a merge mirrors, the rest are
// half-cleaners), so virtual +inf padding above n never moves and comparators reaching beyond n are skipped.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void bitonic_sort(uint64_t* s, int n, int tid, int nthreads) {
  int P = 1;
  while (P < n) P <<= 1;
  for (int k = 2; k <= P; k <<= 1) {
    const int hk = k >> 1;
    for (int t = tid; t < (P >> 1); t += nthreads) {
      const int off = t & (hk - 1), b0 = (t - off) << 1;  // b0 = (t / hk) * k
      const int i = b0 + off, l = b0 + (k - 1 - off);
      if (l < n) {
        const uint64_t a = s[i], b = s[l];
        if (a > b) { s[i] = b; s[l] = a; }
      }
    }
    __syncthreads();
    for (int j = k >> 2; j > 0; j >>= 1) {
      for (int t = tid; t < (P >> 1); t += nthreads) {
        const int off = t & (j - 1);
        const int i = ((t - off) << 1) + off, l = i + j;
        if (l < n) {
          const uint64_t a = s[i], b = s[l];
          if (a > b) { s[i] = b; s[l] = a; }
        }
      }
      __syncthreads();
    }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// Register-resident bitonic network (evidence: profiles/r1_v3_regions.md -- a shared-memory network with one
// __syncthreads per level took 38.6 + 21.8 us).  A bucket of up to 32 * E * NW keys is held by NW warps, E consecutive
// keys per thread: strides below E are in-register compare-exchanges, strides E .. 16 E are SHFL.XOR exchanges, and
// only strides >= 32 E (none for NW = 1) go through shared memory with a barrier.  Normalised network: every
// comparator is ascending; the first step of a K-merge pairs i with its mirror i ^ (K - 1), the other steps i with
// i ^ j.  The (K, j) loops are run-time loops around unrolled per-stride bodies (fully unrolled, the network is
// ~160 KB of straight-line code and runs at the instruction-fetch rate).  Padding keys are +inf.
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void cmp_swap(uint64_t& a, uint64_t& b) {
  const bool sw = a > b;
  const uint64_t lo = sw ? b : a, hi = sw ? a : b;
  a = lo; b = hi;
}

// in-register comparators between e and e ^ X for every e whose bit B is clear (X = B: half-cleaner, X = 2B - 1: mirror)
template <int E, int B, bool MIRROR>
__device__ __forceinline__ void reg_step(uint64_t (&k)[E]) {
  constexpr int X = MIRROR ? 2 * B - 1 : B;
#pragma unroll
  for (int e = 0; e < E; ++e)
    if ((e & B) == 0) cmp_swap(k[e], k[e ^ X]);
}

template <int E, bool MIRROR>
__device__ __forceinline__ void reg_step_dyn(uint64_t (&k)[E], int B) {
  if (E > 1 && B == 1) reg_step<E, 1, MIRROR>(k);
  if (E > 2 && B == 2) reg_step<E, (E > 2 ? 2 : 1), MIRROR>(k);
  if (E > 4 && B == 4) reg_step<E, (E > 4 ? 4 : 1), MIRROR>(k);
  if (E > 8 && B == 8) reg_step<E, (E > 8 ? 8 : 1), MIRROR>(k);
}

// cross-lane step: partner lane = lane ^ d; `lower` threads keep the minima
template <int E, bool MIRROR>
__device__ __forceinline__ void lane_step(uint64_t (&k)[E], int d, bool lower) {
  uint64_t o[E];
#pragma unroll
  for (int e = 0; e < E; ++e) o[e] = __shfl_xor_sync(0xffffffffu, k[MIRROR ? E - 1 - e : e], d);
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const bool take = (o[e] < k[e]) == lower;
    k[e] = take ? o[e] : k[e];
  }
}

// cross-warp step through shared memory, layout s[e * T + tid] (conflict-free for the store and the partner load)
template <int E, int T, bool MIRROR>
__device__ __forceinline__ void smem_step(uint64_t (&k)[E], uint64_t* s, int tid, int x, bool lower) {
#pragma unroll
  for (int e = 0; e < E; ++e) s[e * T + tid] = k[e];
  __syncthreads();
  const int pt = tid ^ x;
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const uint64_t o = s[(MIRROR ? E - 1 - e : e) * T + pt];
    const bool take = (o < k[e]) == lower;
    k[e] = take ? o : k[e];
  }
  __syncthreads();
}

// What the compositing kernels read for a sorted key (.. | index << 8 | mask): the list entry (visible slot << 8 | region
// mask) and the instance's whitened tile-local offset (u0, v0) = -L^T (mean - tile origin), in fp64 (gs_raster.cuh).
struct SortOut {
  float4* rec;   // {u0, v0, bits(slot << 8 | mask), -} per sorted instance
  const uint32_t* slot_of;
  const float4* feat;
  int ox, oy;  // pixel origin of the bucket's tile
};

__device__ __forceinline__ void write_entry(const SortOut& o, int i, uint64_t key) {
  const uint32_t lo = (uint32_t)key;
  const uint32_t slot = __ldg(o.slot_of + (lo >> 8));
  const float4 f0 = __ldg(o.feat + 3 * (size_t)slot), f1 = __ldg(o.feat + 3 * (size_t)slot + 1);
  float u0, v0, mx, my;
  decode_whitened(f0, f1, o.ox, o.oy, u0, v0, mx, my);
  o.rec[i] = make_float4(u0, v0, __uint_as_float((slot << 8) | (lo & 0xffu)), 0.f);
}

template <int E, int NW>
__device__ __forceinline__ void bucket_sort(uint64_t* __restrict__ g, const SortOut& out, int n, uint64_t* s, int tid) {
  constexpr int T = 32 * NW;
  uint64_t k[E];
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = tid * E + e;
    k[e] = i < n ? g[i] : ~0ull;
  }
  int P = 64;
  while (P < n) P <<= 1;  // merges beyond the first power of two >= n would only move padding
#pragma unroll 1
  for (int K = 2; K <= P; K <<= 1) {
    if (K <= E) reg_step_dyn<E, true>(k, K >> 1);
    else if (NW == 1 || K <= 32 * E) lane_step<E, true>(k, K / E - 1, (tid & (K / (2 * E))) == 0);
    else smem_step<E, T, true>(k, s, tid, K / E - 1, (tid & (K / (2 * E))) == 0);
#pragma unroll 1
    for (int j = K >> 2; j >= 1; j >>= 1) {
      if (NW > 1 && j >= 32 * E) smem_step<E, T, false>(k, s, tid, j / E, (tid & (j / E)) == 0);
      else if (j >= E) lane_step<E, false>(k, j / E, (tid & (j / E)) == 0);
      else reg_step_dyn<E, false>(k, j);
    }
  }
  // epilogue in phases of up to four keys, so that the dependent gather chains (key -> slot -> feature record) of a
  // thread overlap without holding E feature records in registers
  constexpr int C = E < 4 ? E : 4;
#pragma unroll
  for (int c = 0; c < E; c += C) {
    uint32_t slot[C];
    float4 f0[C], f1[C];
#pragma unroll
    for (int e = 0; e < C; ++e) slot[e] = (tid * E + c + e < n) ? __ldg(out.slot_of + ((uint32_t)k[c + e] >> 8)) : 0u;
#pragma unroll
    for (int e = 0; e < C; ++e) {
      f0[e] = __ldg(out.feat + 3 * (size_t)slot[e]);
      f1[e] = __ldg(out.feat + 3 * (size_t)slot[e] + 1);
    }
#pragma unroll
    for (int e = 0; e < C; ++e) {
      const int i = tid * E + c + e;
      if (i < n) {
        g[i] = k[c + e];
        float u0, v0, mx, my;
        decode_whitened(f0[e], f1[e], out.ox, out.oy, u0, v0, mx, my);
        out.rec[i] = make_float4(u0, v0, __uint_as_float((slot[e] << 8) | ((uint32_t)k[c + e] & 0xffu)), 0.f);
      }
    }
  }
}


// Buckets of 2048 .. kLargeSort keys (the first n_large entries of `order`): one CTA of 512 threads per bucket, 16 keys
// per thread; beyond kLargeSort the shared-memory-free network above runs in place in global memory (slow; degenerate
// scenes only).
__global__ void __launch_bounds__(512)
tile_sort_large_kernel(int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                       const Counts* __restrict__ counts, uint64_t* __restrict__ keys,
                       float4* __restrict__ rec, const uint32_t* __restrict__ slot_of, const float4* __restrict__ feat) {
  extern __shared__ uint64_t s_dyn[];
  const int tid = threadIdx.x, nth = blockDim.x;
  const int limit = (int)counts->n_large;
  for (int b = blockIdx.x; b < limit; b += gridDim.x) {
    const int tile = (int)order[b];
    const uint2 r = ranges[tile];
    const int n = (int)(r.y - r.x);
    if (n <= kMidSortMax) continue;
    uint64_t* g = keys + r.x;
    const SortOut out = {rec + r.x, slot_of, feat, (tile % tiles_x) * GS_TILE, (tile / tiles_x) * GS_TILE};
    if (n > kLargeSort) {
      bitonic_sort(g, n, tid, nth);  // __syncthreads orders the CTA's own global writes
      for (int t = tid; t < n; t += nth) write_entry(out, t, g[t]);
      __syncthreads();
      continue;
    }
    if (n <= 4096) bucket_sort<8, 16>(g, out, n, s_dyn, tid);
    else bucket_sort<16, 16>(g, out, n, s_dyn, tid);
    __syncthreads();
  }
}

// Buckets up to kMidSortMax keys.  CTAs of 4 warps: the first n_mid entries of `order` (256 .. 2047 keys; those of the
// large kernel are skipped) take a whole CTA each, 8 keys per thread; the remaining buckets (< 256 keys) take one warp
// each, four buckets per CTA, no barrier at all.
// (an explicit minimum of 1 CTA per SM lets ptxas take 110 registers instead of 92: four of these CTAs then no longer fit
// beside the 512-thread CTA of tile_sort_large_kernel, and the two kernels of a scene with long buckets ran one after the other)
#ifdef GS_SORT_MIN_CTAS
__global__ void __launch_bounds__(128, GS_SORT_MIN_CTAS)
#else
__global__ void __launch_bounds__(128)
#endif
tile_sort_kernel(int tiles, int tiles_x, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                 const Counts* __restrict__ counts, uint64_t* __restrict__ keys,
                 float4* __restrict__ rec, const uint32_t* __restrict__ slot_of, const float4* __restrict__ feat,
                 bool do_large) {
  __shared__ uint64_t s_x[2048];
  const int tid = threadIdx.x;
  pdl_enter();
  const int n_mid = (int)counts->n_mid;
  if ((int)blockIdx.x < n_mid) {
    const int tile = (int)order[blockIdx.x];
    const uint2 r = ranges[tile];
    const int n = (int)(r.y - r.x);
    const SortOut out = {rec + r.x, slot_of, feat, (tile % tiles_x) * GS_TILE, (tile / tiles_x) * GS_TILE};
    if (n > kMidSortMax) {
      // a long bucket: tile_sort_large_kernel's, unless the host did not launch it (do_large: the last finished iteration
      // had no long bucket, so the side-stream launch was skipped) -- then sorted here in global memory: slow, correct, and
      // the next iteration launches the large kernel again
      if (do_large) {
        bitonic_sort(keys + r.x, n, tid, 128);
        for (int t = tid; t < n; t += 128) write_entry(out, t, keys[r.x + t]);
      }
      return;
    }
    // keys per thread matched to the bucket: the network runs over 128 E slots whatever n is
    if (n <= 512) bucket_sort<4, 4>(keys + r.x, out, n, s_x, tid);
    else if (n <= 1024) bucket_sort<8, 4>(keys + r.x, out, n, s_x, tid);
    else bucket_sort<16, 4>(keys + r.x, out, n, s_x, tid);
    return;
  }
  const int idx = n_mid + ((int)blockIdx.x - n_mid) * 4 + (tid >> 5);
  if (idx >= tiles) return;
  const int tile = (int)order[idx];
  const uint2 r = ranges[tile];
  const int n = (int)(r.y - r.x), lane = tid & 31;
  if (n == 0) return;
  const SortOut out = {rec + r.x, slot_of, feat, (tile % tiles_x) * GS_TILE, (tile / tiles_x) * GS_TILE};
  if (n <= 64) bucket_sort<2, 1>(keys + r.x, out, n, nullptr, lane);
  else if (n <= 128) bucket_sort<4, 1>(keys + r.x, out, n, nullptr, lane);
  else bucket_sort<8, 1>(keys + r.x, out, n, nullptr, lane);
}

// export for gs_get_binning: keys_sorted[k] = tile << 32 | depth bits
__global__ void export_keys_kernel(int tiles, const uint2* __restrict__ ranges, const uint64_t* __restrict__ keys,
                                   uint64_t* __restrict__ out) {
  const int tile = blockIdx.x;
  if (tile >= tiles) return;
  const uint2 r = ranges[tile];
  for (uint32_t k = r.x + threadIdx.x; k < r.y; k += blockDim.x) out[k] = ((uint64_t)tile << 32) | (keys[k] >> 32);
}

__global__ void export_ids_kernel(int tiles, const uint2* __restrict__ ranges, const float4* __restrict__ rec,
                                  const uint32_t* __restrict__ vis_ids, uint32_t* __restrict__ out) {
  const int tile = blockIdx.x;
  if (tile >= tiles) return;
  const uint2 r = ranges[tile];  // per tile range: in exact-cull mode the entries between two lists are unspecified
  for (uint32_t k = r.x + threadIdx.x; k < r.y; k += blockDim.x) out[k] = vis_ids[__float_as_uint(rec[k].z) >> 8];  // slot -> Gaussian index
}

int export_sorted_ids(gs_ctx* ctx, cudaStream_t s, int64_t I, uint32_t* out) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (I <= 0 || tiles == 0) return GS_OK;
  export_ids_kernel<<<tiles, 128, 0, s>>>(tiles, ctx->ranges, ctx->inst_rec, ctx->vis_ids, out);
  GS_LAUNCH_CHECK("export_ids_kernel");
  return GS_OK;
}

int export_sorted_keys(gs_ctx* ctx, cudaStream_t s, uint64_t* out) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (tiles == 0) return GS_OK;
  export_keys_kernel<<<tiles, 128, 0, s>>>(tiles, ctx->ranges, ctx->keys[0], out);
  GS_LAUNCH_CHECK("export_keys_kernel");
  return GS_OK;
}

int ensure_instance_capacity(gs_ctx* ctx, int64_t need) {
  if (need <= ctx->cap_I) return GS_OK;
  GS_CUDA(cudaDeviceSynchronize());
  const int64_t cap = need + need / 4 + 4096;
  if (cap >= (1ll << 31)) return fail(ctx, GS_E_NOMEM, "more than 2^31 tile instances");
  int rc;
  if ((rc = grow(ctx, ctx->keys[0], cap)) != GS_OK) return rc;
  if ((rc = grow(ctx, ctx->inst_rec, cap)) != GS_OK) return rc;
  ctx->cap_I = cap;
  return GS_OK;
}

// If the mailbox shows that an earlier asynchronous iteration overflowed: grow to fit it, clear the flag and return
// GS_E_OVERFLOW (the caller re-issues the iteration), or GS_E_NOMEM if the scratch could not grow (the old buffers and
// capacity stay valid, the flag stays set).  GS_OK when nothing overflowed.
int handle_overflow(gs_ctx* ctx) {
  const Counts mb = read_mailbox(ctx);
  if (!mb.overflow) return GS_OK;
  const int rc = ensure_instance_capacity(ctx, (int64_t)mb.n_instances + (int64_t)mb.n_instances / 4);
  if (rc != GS_OK) return rc;
  ctx->mailbox->overflow = 0;
  return fail(ctx, GS_E_OVERFLOW, "tile-instance capacity exceeded in an earlier iteration; scratch has grown, re-issue");
}

static int run_tile_scan(gs_ctx* ctx, cudaStream_t s, bool clear) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  if (tiles == 0) return GS_OK;
  if (!ctx->scan_ws) {
    GS_CUDA(cudaMalloc((void**)&ctx->scan_ws, (size_t)kScanMaxCta * kScanAgg * sizeof(unsigned long long)));
    GS_CUDA(cudaMemset(ctx->scan_ws, 0, (size_t)kScanMaxCta * kScanAgg * sizeof(unsigned long long)));
  }
  uint32_t* agg = ctx->scan_ws;
  uint32_t* flags = nullptr;  // (unused: the epoch travels inside the totals)
  const uint32_t epoch = ++ctx->scan_epoch;
  const int nb1 = (int)div_up(tiles, kScanT);
  const int nb8 = (int)div_up(tiles, kScanT * 8);
  if (nb8 > kScanMaxCta) return fail(ctx, GS_E_INVALID, "gs_bin_tiles: more than 262144 tiles");
  int tiles_arg = tiles;
  uint32_t* count_arg = ctx->tile_count;
  Counts* next_arg = clear ? reinterpret_cast<Counts*>(ctx->hdr + 64 * ((ctx->seq + 1u) & 1u)) : nullptr;
  int64_t cap_arg = ctx->cap_I;
  uint32_t seq_arg = ctx->seq, epoch_arg = epoch;
  void* args[] = {&tiles_arg, &count_arg, &ctx->tile_cursor, &ctx->ranges, &ctx->tile_order, &agg, &flags, &epoch_arg,
                  &cap_arg, &ctx->counts, &ctx->mailbox_dev, &seq_arg, &next_arg};
  // cooperative launch: co-residency of the CTAs that wait on each other's flags is guaranteed by the runtime; the
  // programmatic-serialization attribute (pdl_enter) is added when the driver accepts the combination
  const void* fn = nb1 <= kScanMaxCta ? (const void*)tile_scan_kernel<1> : (const void*)tile_scan_kernel<8>;
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(nb1 <= kScanMaxCta ? nb1 : nb8); cfg.blockDim = dim3(kScanT); cfg.stream = s;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeCooperative; at[0].val.cooperative = 1;
  at[1].id = cudaLaunchAttributeProgrammaticStreamSerialization; at[1].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = ctx->scan_pdl ? 2 : 1;
  cudaError_t e = cudaLaunchKernelExC(&cfg, fn, args);
  if (e != cudaSuccess && ctx->scan_pdl) {
    cudaGetLastError();
    ctx->scan_pdl = false;
    cfg.numAttrs = 1;
    e = cudaLaunchKernelExC(&cfg, fn, args);
  }
  GS_CUDA(e);
  if (clear) {  // the scan leaves the counters of THIS image size zero
    ctx->hdr_clean = true;
    if (ctx->ctr_dirty <= (int64_t)tiles) ctx->ctr_dirty = 0;
  }
  GS_LAUNCH_CHECK("tile_scan_kernel");
  return GS_OK;
}

int launch_binning(gs_ctx* ctx, cudaStream_t s) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  GS_PROF(2, s);
  const bool same_shape = ctx->calibrated && ctx->cal_N == ctx->N && ctx->cal_W == ctx->cam.W && ctx->cal_H == ctx->cam.H;
  int rc;
  if (!same_shape) {
    // calibration: scan the tile counts, read the instance total, size the buffers, scan again if it was short.
    // This is the only synchronising path of the iteration.
    if ((rc = run_tile_scan(ctx, s, false)) != GS_OK) return rc;
    GS_CUDA(cudaStreamSynchronize(s));
    const int64_t I = ctx->mailbox->n_instances;
    if (I > ctx->cap_I) {
      if ((rc = ensure_instance_capacity(ctx, I)) != GS_OK) return rc;
      if ((rc = run_tile_scan(ctx, s, false)) != GS_OK) return rc;
    }
    ctx->mailbox->overflow = 0;
    ctx->calibrated = true;
    ctx->cal_N = ctx->N; ctx->cal_W = ctx->cam.W; ctx->cal_H = ctx->cam.H;
  } else {
    // asynchronous path: act on what the last finished iteration reported (no synchronisation): an overflow is
    // reported to the caller (after growing), a near-full buffer is grown ahead of time
    if ((rc = handle_overflow(ctx)) != GS_OK) return rc;
    const Counts mb = read_mailbox(ctx);
    if ((int64_t)mb.n_instances + (int64_t)mb.n_instances / 8 > ctx->cap_I)
      if ((rc = ensure_instance_capacity(ctx, (int64_t)mb.n_instances + (int64_t)mb.n_instances / 4)) != GS_OK) return rc;
    if ((rc = run_tile_scan(ctx, s, true)) != GS_OK) return rc;
  }
  GS_PROF(3, s);
  if (ctx->N > 0) {
    // grid: enough CTAs for 1.5 x the visible count of the last finished iteration (the kernel strides over the rest)
    const int64_t v_hint = (int64_t)read_mailbox(ctx).n_visible;
    const int64_t emit_ctas = std::min<int64_t>(div_up(ctx->N, kEmitG), std::max<int64_t>(div_up(v_hint + v_hint / 2, kEmitG), 148 * 8));
    GS_LAUNCH_PDL(emit_kernel, (unsigned)emit_ctas, kEmitT, 0, s, (const uint4*)ctx->vis_rec,
                  (const float4*)ctx->feat, ctx->cam.tiles_x, ctx->tile_cursor, (const Counts*)ctx->counts, ctx->keys[0],
                  ctx->opt_exact_cull);
    GS_LAUNCH_CHECK("emit_kernel");
    if (ctx->opt_exact_cull && tiles > 0) {
      GS_LAUNCH_PDL(range_fix_kernel, (unsigned)div_up(tiles, 256), 256, 0, s, tiles, (const uint32_t*)ctx->tile_cursor, ctx->ranges);
      GS_LAUNCH_CHECK("range_fix_kernel");
    }
  }
  GS_PROF(4, s);
  if (ctx->N > 0 && tiles > 0) {
    if (!ctx->sort_attr_set) {
      GS_CUDA(cudaFuncSetAttribute(tile_sort_large_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   kLargeSort * (int)sizeof(uint64_t)));
      ctx->sort_attr_set = true;
    }
    // The few long buckets (block-wide network) sort on the side stream while the warp kernel sorts the rest -- when there
    // are any: the number of long buckets of the last finished iteration (mailbox; exact after a calibration pass) decides
    // whether the side-stream kernel is launched at all.  Without it the main stream is one chain of programmatically
    // dependent kernels; a long bucket that shows up unannounced is sorted by tile_sort_kernel itself (slow path).
    const bool large = ctx->side_stream != nullptr && read_mailbox(ctx).n_large > 0;
    if (large) {
      cudaStream_t sl = ctx->side_stream;
      GS_CUDA(cudaEventRecord(ctx->ev_fork2, s));
      GS_CUDA(cudaStreamWaitEvent(sl, ctx->ev_fork2, 0));
      tile_sort_large_kernel<<<min(tiles, 296), 512, kLargeSort * sizeof(uint64_t), sl>>>(
          ctx->cam.tiles_x, ctx->tile_order, ctx->ranges, ctx->counts, ctx->keys[0], ctx->inst_rec, ctx->slot_of,
          ctx->feat);
      GS_LAUNCH_CHECK("tile_sort_large_kernel");
      GS_CUDA(cudaEventRecord(ctx->ev_join2, sl));
    }
    GS_LAUNCH_PDL(tile_sort_kernel, tiles, 128, 0, s, tiles, ctx->cam.tiles_x, (const uint32_t*)ctx->tile_order,
                  (const uint2*)ctx->ranges, (const Counts*)ctx->counts, ctx->keys[0], ctx->inst_rec,
                  (const uint32_t*)ctx->slot_of, (const float4*)ctx->feat, !large);
    GS_LAUNCH_CHECK("tile_sort_kernel");
    if (large) GS_CUDA(cudaStreamWaitEvent(s, ctx->ev_join2, 0));
  }
  ctx->sorted_buf = 0;
  GS_PROF(5, s);
  return GS_OK;
}

}  // namespace gs
