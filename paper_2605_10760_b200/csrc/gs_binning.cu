// gs_binning.cu -- steps a2-a5: per-tile instance lists ordered by (depth key, Gaussian index).
//
// Design (evidence: profiles/r1_v1_baseline.md -- a 6-pass one-sweep LSD radix sort of 64-bit (tile << 32 | depth)
// keys plus a serial per-thread duplication cost 112 + 40 us of a 614 us iteration): the sort on (tile, depth, index)
// keys is split MSD-first.
//   1. gs_preprocess counts the instances of every tile (atomics on tile_count) while it computes the rects.
//   2. tile_scan_kernel (one CTA): exclusive prefix sum over the tile counts = the per-tile ranges (step a5 comes for
//      free), the instance total / overflow flag, and the tile order by descending list length.
//   3. emit_kernel: every visible Gaussian appends (depth bits << 32 | index) to the bucket of each tile of its rect
//      (atomic cursor per tile) -- a counting-sort pass on the tile digit; the order inside a bucket is arbitrary.
//   4. tile_sort_kernel: every bucket is sorted by its 64-bit key in shared memory (bitonic network).  The keys are
//      unique (the index is part of the key), so the result is THE (tile, depth bits, index) order, bit for bit,
//      whatever the arrival order was.  Buckets beyond the shared-memory capacity are sorted in global memory.
// Integer work only.  Bytes: 8 I (emit) + 8 I (sort read) + 12 I (sorted keys + ids) vs (8 + 24 * 6) I before.
#include "gs_internal.cuh"

namespace gs {

constexpr int kSmallSortMax = 255;  // buckets up to this size are sorted by one warp (whole length/8 classes of the tile order)
constexpr int kMidSortMax = 1023;   // buckets up to this size are sorted by one CTA of 4 warps; beyond: the large kernel
constexpr int kLargeSort = 8192;
constexpr int kScanCache = 8192;   // tile counts cached in shared memory by the scan kernel (all of them up to ~2 Mpix)
// tile_count / tile_cursor are strided by 32 words: one counter per 128-byte line, so that the atomics of different
// tiles are served by different L2 lines (3225 adjacent counters would share ~100 lines and serialise there)   // up to this size: 512-thread CTA, 64 KB dynamic shared memory; beyond: global memory

// ---------------------------------------------------------------------------------------------------------------
// a2 + a5: prefix sum over the tile counts, ranges, totals, overflow flag, LPT tile order.  One CTA of 1024 threads.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024)
tile_scan_kernel(int tiles, const uint32_t* __restrict__ tile_count, uint32_t* __restrict__ tile_cursor,
                 uint2* __restrict__ ranges, uint32_t* __restrict__ order, int64_t capacity, Counts* counts,
                 Counts* mailbox, uint32_t seq) {
  __shared__ uint32_t hist[1024];
  __shared__ uint32_t wsum[32];
  __shared__ uint32_t s_carry, s_large, s_mid;
  __shared__ uint32_t s_cnt[kScanCache];  // the counts, fetched once with all loads in flight together
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int t = tid; t < min(tiles, kScanCache); t += 1024) s_cnt[t] = tile_count[(size_t)t * kCtrStride];
  hist[tid] = 0;
  if (tid == 0) { s_carry = 0; s_large = 0; s_mid = 0; }
  __syncthreads();
  // exclusive scan of the counts, 1024 tiles per round
  for (int base = 0; base < tiles; base += 1024) {
    const int t = base + tid;
    const uint32_t c = t < tiles ? (t < kScanCache ? s_cnt[t] : tile_count[(size_t)t * kCtrStride]) : 0u;
    uint32_t incl = c;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
      if (lane >= d) incl += v;
    }
    if (lane == 31) wsum[warp] = incl;
    __syncthreads();
    uint32_t off = s_carry + incl - c;
    for (int w = 0; w < warp; ++w) off += wsum[w];
    if (t < tiles) {
      tile_cursor[(size_t)t * kCtrStride] = off;
      ranges[t] = c ? make_uint2(off, off + c) : make_uint2(0u, 0u);  // cleared below if the iteration overflows
      atomicAdd(&hist[1023 - min(c >> 3, 1023u)], 1u);
      if (c > (uint32_t)kMidSortMax) atomicAdd(&s_large, 1u);
      if (c > (uint32_t)kSmallSortMax) atomicAdd(&s_mid, 1u);
    }
    __syncthreads();
    if (tid == 1023) s_carry = off + c;
    __syncthreads();
  }
  const uint32_t I = s_carry;
  const bool ovf = (int64_t)I > capacity;
  if (tid == 0) {
    counts->n_instances = I;
    counts->overflow = ovf ? 1u : 0u;
    counts->n_large = s_large;
    counts->n_mid = s_mid;
    counts->seq = seq;
    mailbox->n_instances = I;
    mailbox->overflow = ovf ? 1u : 0u;
    mailbox->n_visible = counts->n_visible;
    __threadfence_system();
    mailbox->seq = seq;
  }
  if (ovf)
    for (int t = tid; t < tiles; t += 1024) ranges[t] = make_uint2(0u, 0u);  // the flagged iteration renders nothing
  // tile ids by descending list length (counting sort on length / 8; order inside a bucket is arbitrary)
  const uint32_t h = hist[tid];
  uint32_t incl = h;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  __syncthreads();
  if (lane == 31) wsum[warp] = incl;
  __syncthreads();
  uint32_t bbase = incl - h;
  for (int w = 0; w < warp; ++w) bbase += wsum[w];
  __syncthreads();
  hist[tid] = bbase;
  __syncthreads();
  for (int t = tid; t < tiles; t += 1024)
    order[atomicAdd(&hist[1023 - min((t < kScanCache ? s_cnt[t] : tile_count[(size_t)t * kCtrStride]) >> 3, 1023u)], 1u)] = (uint32_t)t;
}

// ---------------------------------------------------------------------------------------------------------------
// a3: duplication.  One thread per Gaussian; (depth bits << 32 | index) goes to the bucket of every tile of the rect.
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
emit_kernel(const uint32_t* __restrict__ vis_ids, const uint32_t* __restrict__ tiles_touched, const ushort4* __restrict__ rect,
            const uint32_t* __restrict__ depth_key, int tiles_x, uint32_t* __restrict__ tile_cursor,
            const Counts* __restrict__ counts, uint64_t* __restrict__ keys) {
  // Block-cooperative: the instances of the block's 256 Gaussians form one work list (prefix sum of the per-Gaussian
  // tile counts); every round the 256 threads take 256 consecutive work items, whatever Gaussian they belong to, so a
  // Gaussian covering hundreds of tiles is emitted by the whole block; four independent atomics per thread are put in
  // flight before their results are used.
  __shared__ uint32_t s_excl[257], s_w[256], s_xy[256], s_ws[8];
  __shared__ uint64_t s_key[256];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (counts->overflow) return;
  const uint32_t V = counts->n_visible;
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + tid;
  if ((int64_t)blockIdx.x * blockDim.x >= (int64_t)V) return;
  const uint32_t i = (k < V) ? vis_ids[k] : 0u;
  const uint32_t n = (k < V) ? tiles_touched[i] : 0u;
  ushort4 r = make_ushort4(0, 0, 1, 0);
  uint64_t key = 0;
  if (n) {
    r = rect[i];
    key = ((uint64_t)depth_key[i] << 32) | (uint64_t)i;
  }
  uint32_t incl = n;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) s_ws[warp] = incl;
  __syncthreads();
  uint32_t wb = 0;
#pragma unroll
  for (int q = 0; q < 8; ++q) wb += (q < warp) ? s_ws[q] : 0u;
  s_excl[tid] = wb + incl - n;
  s_w[tid] = (uint32_t)(r.z - r.x);
  s_xy[tid] = (uint32_t)r.x | ((uint32_t)r.y << 16);
  s_key[tid] = key;
  if (tid == 255) s_excl[256] = wb + incl;
  __syncthreads();
  const uint32_t total = s_excl[256];
  for (uint32_t base = 0; base < total; base += 1024) {
    uint32_t* cur[4];
    uint64_t kk[4];
    uint32_t pos[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const uint32_t item = base + u * 256 + tid;
      cur[u] = nullptr;
      if (item < total) {
        int owner = 0;  // last Gaussian of the block whose exclusive prefix is <= item
#pragma unroll
        for (int step = 128; step >= 1; step >>= 1)
          if (s_excl[owner + step] <= item) owner += step;
        const uint32_t local = item - s_excl[owner], w = s_w[owner], xy = s_xy[owner];
        const uint32_t ty = (xy >> 16) + local / w, tx = (xy & 0xffffu) + local % w;
        cur[u] = &tile_cursor[(size_t)(ty * tiles_x + tx) * kCtrStride];
        kk[u] = s_key[owner];
      }
    }
#pragma unroll
    for (int u = 0; u < 4; ++u) pos[u] = cur[u] ? atomicAdd(cur[u], 1u) : 0u;
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (cur[u]) keys[pos[u]] = kk[u];
  }
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

template <int E, int NW>
__device__ __forceinline__ void bucket_sort(uint64_t* __restrict__ g, uint32_t* __restrict__ ids, int n, uint64_t* s, int tid) {
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
#pragma unroll
  for (int e = 0; e < E; ++e) {
    const int i = tid * E + e;
    if (i < n) { g[i] = k[e]; ids[i] = (uint32_t)k[e]; }
  }
}

// Buckets of 1024 .. kLargeSort keys (the first n_large entries of `order`): one CTA of 512 threads per bucket, 16 keys
// per thread; beyond kLargeSort the shared-memory-free network above runs in place in global memory (slow; degenerate
// scenes only).
__global__ void __launch_bounds__(512)
tile_sort_large_kernel(const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                       const Counts* __restrict__ counts, uint64_t* __restrict__ keys, uint32_t* __restrict__ ids) {
  extern __shared__ uint64_t s_dyn[];
  const int tid = threadIdx.x, nth = blockDim.x;
  const int limit = (int)counts->n_large;
  for (int b = blockIdx.x; b < limit; b += gridDim.x) {
    const int tile = (int)order[b];
    const uint2 r = ranges[tile];
    const int n = (int)(r.y - r.x);
    if (n <= kMidSortMax) continue;
    uint64_t* g = keys + r.x;
    if (n > kLargeSort) {
      bitonic_sort(g, n, tid, nth);  // __syncthreads orders the CTA's own global writes
      for (int t = tid; t < n; t += nth) ids[r.x + t] = (uint32_t)g[t];
      __syncthreads();
      continue;
    }
    if (n <= 2048) bucket_sort<4, 16>(g, ids + r.x, n, s_dyn, tid);
    else bucket_sort<16, 16>(g, ids + r.x, n, s_dyn, tid);
    __syncthreads();
  }
}

// Buckets up to kMidSortMax keys.  CTAs of 4 warps: the first n_mid entries of `order` (256 .. 1023 keys; those of the
// large kernel are skipped) take a whole CTA each, 8 keys per thread; the remaining buckets (< 256 keys) take one warp
// each, four buckets per CTA, no barrier at all.
__global__ void __launch_bounds__(128)
tile_sort_kernel(int tiles, const uint32_t* __restrict__ order, const uint2* __restrict__ ranges,
                 const Counts* __restrict__ counts, uint64_t* __restrict__ keys, uint32_t* __restrict__ ids) {
  __shared__ uint64_t s_x[1024];
  const int tid = threadIdx.x;
  const int n_mid = (int)counts->n_mid;
  if ((int)blockIdx.x < n_mid) {
    const uint2 r = ranges[order[blockIdx.x]];
    const int n = (int)(r.y - r.x);
    if (n > kMidSortMax) return;
    bucket_sort<8, 4>(keys + r.x, ids + r.x, n, s_x, tid);
    return;
  }
  const int idx = n_mid + ((int)blockIdx.x - n_mid) * 4 + (tid >> 5);
  if (idx >= tiles) return;
  const uint2 r = ranges[order[idx]];
  const int n = (int)(r.y - r.x), lane = tid & 31;
  if (n == 0) return;
  if (n <= 64) bucket_sort<2, 1>(keys + r.x, ids + r.x, n, nullptr, lane);
  else bucket_sort<8, 1>(keys + r.x, ids + r.x, n, nullptr, lane);
}

// export for gs_get_binning: keys_sorted[k] = tile << 32 | depth bits
__global__ void export_keys_kernel(int tiles, const uint2* __restrict__ ranges, const uint64_t* __restrict__ keys,
                                   uint64_t* __restrict__ out) {
  const int tile = blockIdx.x;
  if (tile >= tiles) return;
  const uint2 r = ranges[tile];
  for (uint32_t k = r.x + threadIdx.x; k < r.y; k += blockDim.x) out[k] = ((uint64_t)tile << 32) | (keys[k] >> 32);
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
  if ((rc = grow(ctx, ctx->vals[0], cap)) != GS_OK) return rc;
  ctx->cap_I = cap;
  return GS_OK;
}

// If the mailbox shows that an earlier asynchronous iteration overflowed: grow to fit it, clear the flag, return true.
bool handle_overflow(gs_ctx* ctx) {
  const Counts mb = read_mailbox(ctx);
  if (!mb.overflow) return false;
  ensure_instance_capacity(ctx, (int64_t)mb.n_instances + (int64_t)mb.n_instances / 4);
  ctx->mailbox->overflow = 0;
  return true;
}

static int run_tile_scan(gs_ctx* ctx, cudaStream_t s) {
  const int tiles = ctx->cam.tiles_x * ctx->cam.tiles_y;
  tile_scan_kernel<<<1, 1024, 0, s>>>(tiles, ctx->tile_count, ctx->tile_cursor, ctx->ranges, ctx->tile_order,
                                      ctx->cap_I, ctx->counts, ctx->mailbox_dev, ctx->seq);
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
    if ((rc = run_tile_scan(ctx, s)) != GS_OK) return rc;
    GS_CUDA(cudaStreamSynchronize(s));
    const int64_t I = ctx->mailbox->n_instances;
    if (I > ctx->cap_I) {
      if ((rc = ensure_instance_capacity(ctx, I)) != GS_OK) return rc;
      if ((rc = run_tile_scan(ctx, s)) != GS_OK) return rc;
    }
    ctx->mailbox->overflow = 0;
    ctx->calibrated = true;
    ctx->cal_N = ctx->N; ctx->cal_W = ctx->cam.W; ctx->cal_H = ctx->cam.H;
  } else {
    // asynchronous path: act on what the last finished iteration reported (no synchronisation): an overflow is
    // reported to the caller (after growing), a near-full buffer is grown ahead of time
    if (handle_overflow(ctx)) return fail(ctx, GS_E_OVERFLOW, "tile-instance capacity exceeded in an earlier iteration; scratch has grown, re-issue");
    const Counts mb = read_mailbox(ctx);
    if ((int64_t)mb.n_instances + (int64_t)mb.n_instances / 8 > ctx->cap_I)
      if ((rc = ensure_instance_capacity(ctx, (int64_t)mb.n_instances + (int64_t)mb.n_instances / 4)) != GS_OK) return rc;
    if ((rc = run_tile_scan(ctx, s)) != GS_OK) return rc;
  }
  GS_PROF(3, s);
  if (ctx->N > 0) {
    emit_kernel<<<(unsigned)div_up(ctx->N, 256), 256, 0, s>>>(ctx->vis_ids, ctx->tiles_touched, ctx->rect, ctx->depth_key,
                                                              ctx->cam.tiles_x, ctx->tile_cursor, ctx->counts,
                                                              ctx->keys[0]);
    GS_LAUNCH_CHECK("emit_kernel");
  }
  GS_PROF(4, s);
  if (ctx->N > 0 && tiles > 0) {
    if (!ctx->sort_attr_set) {
      GS_CUDA(cudaFuncSetAttribute(tile_sort_large_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                   kLargeSort * (int)sizeof(uint64_t)));
      ctx->sort_attr_set = true;
    }
    // the few long buckets (block-wide network) sort on the side stream while the warp kernel sorts the rest
    const bool fork = ctx->side_stream != nullptr;
    cudaStream_t sl = fork ? ctx->side_stream : s;
    if (fork) {
      GS_CUDA(cudaEventRecord(ctx->ev_fork2, s));
      GS_CUDA(cudaStreamWaitEvent(sl, ctx->ev_fork2, 0));
    }
    tile_sort_large_kernel<<<min(tiles, 296), 512, kLargeSort * sizeof(uint64_t), sl>>>(ctx->tile_order, ctx->ranges, ctx->counts,
                                                                                        ctx->keys[0], ctx->vals[0]);
    GS_LAUNCH_CHECK("tile_sort_large_kernel");
    if (fork) GS_CUDA(cudaEventRecord(ctx->ev_join2, sl));
    tile_sort_kernel<<<tiles, 128, 0, s>>>(tiles, ctx->tile_order, ctx->ranges, ctx->counts, ctx->keys[0], ctx->vals[0]);
    GS_LAUNCH_CHECK("tile_sort_kernel");
    if (fork) GS_CUDA(cudaStreamWaitEvent(s, ctx->ev_join2, 0));
  }
  ctx->sorted_buf = 0;
  GS_PROF(5, s);
  return GS_OK;
}

}  // namespace gs
