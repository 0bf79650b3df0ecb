// gs_binning.cu -- steps a2-a5: prefix sum of tiles touched + duplication into (tile << 32 | depth bits, id) instances
// (one single-pass kernel with decoupled look-back), stable LSD radix sort (one-sweep: one histogram kernel + one
// scatter kernel per 8-bit digit, chained by decoupled look-back), per-tile ranges.  Integer work only; HBM-bound.
#include "gs_internal.cuh"

namespace gs {

__device__ __forceinline__ uint32_t lanemask_lt() {
  uint32_t m;
  asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m));
  return m;
}

__device__ __forceinline__ uint64_t ld_volatile_u64(const uint64_t* p) {
  uint64_t v;
  asm volatile("ld.volatile.global.u64 %0, [%1];" : "=l"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_volatile_u64(uint64_t* p, uint64_t v) {
  asm volatile("st.volatile.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint32_t ld_volatile_u32(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.volatile.global.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_volatile_u32(uint32_t* p, uint32_t v) {
  asm volatile("st.volatile.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ---------------------------------------------------------------------------------------------------------------
// a2 + a3: exclusive scan of tiles_touched (chained scan, status word = flag << 32 | value) and key emission.
// Instances of Gaussian i are emitted ty-major / tx-minor over its tile rect, in ascending i, so a stable sort leaves
// equal (tile, depth) keys in ascending Gaussian index (Q13).
// ---------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kScanThreads)
scan_dup_kernel(int64_t N, const uint32_t* __restrict__ tiles_touched, const ushort4* __restrict__ rect,
                const uint32_t* __restrict__ depth_key, uint64_t* status, uint32_t* ticket, int64_t capacity,
                int tiles_x, uint64_t* __restrict__ keys, uint32_t* __restrict__ vals, Counts* counts,
                Counts* mailbox, uint32_t seq) {
  __shared__ uint32_t s_chunk, s_prefix;
  __shared__ uint32_t s_warp[kScanThreads / 32];
  if (threadIdx.x == 0) s_chunk = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t chunk = s_chunk;
  const int64_t base = (int64_t)chunk * kScanChunk + (int64_t)threadIdx.x * kScanIPT;
  uint32_t cnt[kScanIPT];
  if (base + kScanIPT <= N) {
    const uint4 v = *reinterpret_cast<const uint4*>(tiles_touched + base);
    cnt[0] = v.x; cnt[1] = v.y; cnt[2] = v.z; cnt[3] = v.w;
  } else {
#pragma unroll
    for (int k = 0; k < kScanIPT; ++k) cnt[k] = (base + k < N) ? tiles_touched[base + k] : 0u;
  }
  const uint32_t tsum = cnt[0] + cnt[1] + cnt[2] + cnt[3];
  // block exclusive scan of tsum
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint32_t incl = tsum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t t = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += t;
  }
  if (lane == 31) s_warp[warp] = incl;
  __syncthreads();
  uint32_t wbase = 0, total = 0;
#pragma unroll
  for (int w = 0; w < kScanThreads / 32; ++w) {
    const uint32_t t = s_warp[w];
    if (w < warp) wbase += t;
    total += t;
  }
  if (threadIdx.x == 0) {
    uint32_t prefix = 0;
    if (chunk == 0) {
      st_volatile_u64(status, (2ull << 32) | total);
    } else {
      st_volatile_u64(status + chunk, (1ull << 32) | total);
      int64_t p = (int64_t)chunk - 1;
      while (true) {
        const uint64_t w = ld_volatile_u64(status + p);
        const uint32_t flag = (uint32_t)(w >> 32);
        if (flag == 0) continue;
        prefix += (uint32_t)w;
        if (flag == 2) break;
        --p;
      }
      st_volatile_u64(status + chunk, (2ull << 32) | (uint64_t)(prefix + total));
    }
    s_prefix = prefix;
    const int64_t nchunks = (N + kScanChunk - 1) / kScanChunk;
    if ((int64_t)chunk == nchunks - 1) {
      const uint32_t I = prefix + total;
      const uint32_t ovf = ((int64_t)I > capacity) ? 1u : 0u;
      counts->n_instances = I;
      counts->overflow = ovf;
      counts->seq = seq;
      mailbox->n_instances = I;
      mailbox->overflow = ovf;
      mailbox->n_visible = counts->n_visible;
      __threadfence_system();
      mailbox->seq = seq;
    }
  }
  __syncthreads();
  uint32_t off = s_prefix + wbase + (incl - tsum);
  if ((int64_t)s_prefix + total > capacity) return;  // this block would overrun: the iteration is flagged as overflowed
#pragma unroll
  for (int k = 0; k < kScanIPT; ++k) {
    if (cnt[k] == 0) continue;
    const int64_t i = base + k;
    const ushort4 r = rect[i];
    const uint64_t dk = depth_key[i];
    for (int ty = r.y; ty < r.w; ++ty)
      for (int tx = r.x; tx < r.z; ++tx) {
        keys[off] = ((uint64_t)(uint32_t)(ty * tiles_x + tx) << 32) | dk;
        vals[off] = (uint32_t)i;
        ++off;
      }
  }
}

// ---------------------------------------------------------------------------------------------------------------
// a4: one-sweep LSD radix sort of (u64 key, u32 value) pairs, 8-bit digits, stable.
// ---------------------------------------------------------------------------------------------------------------
struct SortPlan {
  int passes;
  int shift[kMaxPasses];
};

__device__ __forceinline__ uint32_t eff_instances(const Counts* c) { return c->overflow ? 0u : c->n_instances; }

__global__ void __launch_bounds__(kSortThreads)
sort_hist_kernel(const uint64_t* __restrict__ keys, const Counts* __restrict__ counts, SortPlan plan, uint32_t* hist) {
  __shared__ uint32_t sh[kMaxPasses * kRadix];
  const uint32_t I = eff_instances(counts);
  const int64_t base = (int64_t)blockIdx.x * kSortChunk;
  if (base >= I) return;
  for (int k = threadIdx.x; k < plan.passes * kRadix; k += kSortThreads) sh[k] = 0;
  __syncthreads();
#pragma unroll
  for (int j = 0; j < kSortKPT; ++j) {
    const int64_t idx = base + j * kSortThreads + threadIdx.x;
    if (idx < I) {
      const uint64_t key = keys[idx];
      for (int p = 0; p < plan.passes; ++p) atomicAdd(&sh[p * kRadix + (uint32_t)((key >> plan.shift[p]) & (kRadix - 1))], 1u);
    }
  }
  __syncthreads();
  for (int k = threadIdx.x; k < plan.passes * kRadix; k += kSortThreads)
    if (sh[k]) atomicAdd(&hist[k], sh[k]);
}

constexpr uint32_t kFlagAgg = 1u << 30, kFlagIncl = 2u << 30, kValMask = (1u << 30) - 1;

__global__ void __launch_bounds__(kSortThreads)
sort_pass_kernel(const uint64_t* __restrict__ keys_in, const uint32_t* __restrict__ vals_in,
                 uint64_t* __restrict__ keys_out, uint32_t* __restrict__ vals_out, const Counts* __restrict__ counts,
                 int shift, const uint32_t* __restrict__ hist /*[256] of this pass*/, uint32_t* status /*[chunks,256]*/,
                 uint32_t* ticket) {
  __shared__ uint32_t s_chunk;
  __shared__ uint32_t s_whist[kSortThreads / 32][kRadix];
  __shared__ uint32_t s_base[kRadix];
  __shared__ uint32_t s_wsum[kSortThreads / 32];
  if (threadIdx.x == 0) s_chunk = atomicAdd(ticket, 1u);
  __syncthreads();
  const uint32_t chunk = s_chunk;
  const uint32_t I = eff_instances(counts);
  const int64_t base = (int64_t)chunk * kSortChunk;
  if (base >= I) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int k = threadIdx.x; k < (kSortThreads / 32) * kRadix; k += kSortThreads) (&s_whist[0][0])[k] = 0;
  uint64_t key[kSortKPT];
  uint32_t val[kSortKPT], rank[kSortKPT];
  const int64_t wbase = base + (int64_t)warp * (kSortKPT * 32);
#pragma unroll
  for (int j = 0; j < kSortKPT; ++j) {
    const int64_t idx = wbase + j * 32 + lane;
    const bool ok = idx < I;
    key[j] = ok ? keys_in[idx] : ~0ull;
    val[j] = ok ? vals_in[idx] : 0u;
  }
  __syncthreads();
  // stable rank of each key among equal digits inside the block: warp-level match, warps in order
#pragma unroll
  for (int j = 0; j < kSortKPT; ++j) {
    const bool ok = (wbase + j * 32 + lane) < I;
    const uint32_t d = (uint32_t)((key[j] >> shift) & (kRadix - 1));
    const uint32_t tag = ok ? d : (kRadix + lane);
    const uint32_t peers = __match_any_sync(0xffffffffu, tag);
    uint32_t prev = 0;
    if (ok) prev = s_whist[warp][d];
    __syncwarp();
    if (ok && (peers & lanemask_lt()) == 0) s_whist[warp][d] = prev + __popc(peers);
    __syncwarp();
    rank[j] = prev + __popc(peers & lanemask_lt());
  }
  __syncthreads();
  // thread d owns digit d: offsets of the warps inside the block, block count, global base by decoupled look-back
  {
    const int d = threadIdx.x;
    uint32_t run = 0;
#pragma unroll
    for (int w = 0; w < kSortThreads / 32; ++w) {
      const uint32_t t = s_whist[w][d];
      s_whist[w][d] = run;
      run += t;
    }
    // exclusive scan of the global digit histogram (256 values, one per thread)
    const uint32_t h = hist[d];
    uint32_t incl = h;
#pragma unroll
    for (int k = 1; k < 32; k <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, incl, k);
      if (lane >= k) incl += t;
    }
    if (lane == 31) s_wsum[warp] = incl;
    __syncthreads();
    uint32_t gbase = incl - h;
    for (int w = 0; w < warp; ++w) gbase += s_wsum[w];
    uint32_t* st = status + (size_t)chunk * kRadix + d;
    uint32_t acc = 0;
    if (chunk == 0) {
      st_volatile_u32(st, kFlagIncl | run);
    } else {
      st_volatile_u32(st, kFlagAgg | run);
      int64_t q = (int64_t)chunk - 1;
      while (true) {
        const uint32_t w = ld_volatile_u32(status + (size_t)q * kRadix + d);
        if ((w >> 30) == 0) continue;
        acc += w & kValMask;
        if (w & kFlagIncl) break;
        --q;
      }
      st_volatile_u32(st, kFlagIncl | (acc + run));
    }
    s_base[d] = gbase + acc;
  }
  __syncthreads();
#pragma unroll
  for (int j = 0; j < kSortKPT; ++j) {
    if ((wbase + j * 32 + lane) < I) {
      const uint32_t d = (uint32_t)((key[j] >> shift) & (kRadix - 1));
      const uint32_t dst = s_base[d] + s_whist[warp][d] + rank[j];
      keys_out[dst] = key[j];
      vals_out[dst] = val[j];
    }
  }
}

// a5: ranges[t] = [first, last+1) of the sorted instances with tile id t (ranges zeroed beforehand)
__global__ void tile_ranges_kernel(const uint64_t* __restrict__ keys, const Counts* __restrict__ counts,
                                   uint2* __restrict__ ranges) {
  const uint32_t I = eff_instances(counts);
  const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= I) return;
  const uint32_t t = (uint32_t)(keys[k] >> 32);
  if (k == 0 || (uint32_t)(keys[k - 1] >> 32) != t) ranges[t].x = (uint32_t)k;
  if (k == (int64_t)I - 1 || (uint32_t)(keys[k + 1] >> 32) != t) ranges[t].y = (uint32_t)(k + 1);
}

// Tile ids by descending list length (counting sort on length / 8, 1024 buckets; order inside a bucket is arbitrary):
// the compositing kernels launch their regions in this order, so that the longest lists start first (LPT scheduling).
__global__ void __launch_bounds__(1024)
tile_order_kernel(int tiles, const uint2* __restrict__ ranges, uint32_t* __restrict__ order) {
  __shared__ uint32_t hist[1024];
  __shared__ uint32_t wsum[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  hist[tid] = 0;
  __syncthreads();
  for (int t = tid; t < tiles; t += 1024) {
    const uint2 r = ranges[t];
    atomicAdd(&hist[1023 - min((r.y - r.x) >> 3, 1023u)], 1u);
  }
  __syncthreads();
  const uint32_t h = hist[tid];
  uint32_t incl = h;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, incl, d);
    if (lane >= d) incl += v;
  }
  if (lane == 31) wsum[warp] = incl;
  __syncthreads();
  uint32_t base = incl - h;
  for (int w = 0; w < warp; ++w) base += wsum[w];
  __syncthreads();
  hist[tid] = base;  // bucket cursor
  __syncthreads();
  for (int t = tid; t < tiles; t += 1024) {
    const uint2 r = ranges[t];
    order[atomicAdd(&hist[1023 - min((r.y - r.x) >> 3, 1023u)], 1u)] = (uint32_t)t;
  }
}

static int run_scan_dup(gs_ctx* ctx, cudaStream_t s) {
  const int64_t nchunks = div_up(ctx->N, kScanChunk);
  // reset: counts->{n_instances,overflow}, tickets, scan status (n_visible was produced by gs_preprocess: keep it)
  GS_CUDA(cudaMemsetAsync(ctx->scan_status, 0, (size_t)nchunks * sizeof(uint64_t), s));
  GS_CUDA(cudaMemsetAsync(ctx->sort_ticket, 0, (kMaxPasses + 2) * sizeof(uint32_t), s));
  scan_dup_kernel<<<(unsigned)nchunks, kScanThreads, 0, s>>>(ctx->N, ctx->tiles_touched, ctx->rect, ctx->depth_key,
                                                             ctx->scan_status, ctx->sort_ticket + kMaxPasses,
                                                             ctx->cap_I, ctx->cam.tiles_x, ctx->keys[0], ctx->vals[0],
                                                             ctx->counts, ctx->mailbox_dev, ctx->seq);
  GS_LAUNCH_CHECK("scan_dup_kernel");
  return GS_OK;
}

int ensure_instance_capacity(gs_ctx* ctx, int64_t need) {
  if (need <= ctx->cap_I) return GS_OK;
  GS_CUDA(cudaDeviceSynchronize());
  int64_t cap = need + need / 4 + 4096;
  cap = div_up(cap, kSortChunk) * kSortChunk;
  if (cap >= (1ll << 30)) return fail(ctx, GS_E_NOMEM, "more than 2^30 tile instances");
  int rc;
  for (int b = 0; b < 2; ++b) {
    if ((rc = grow(ctx, ctx->keys[b], cap)) != GS_OK) return rc;
    if ((rc = grow(ctx, ctx->vals[b], cap)) != GS_OK) return rc;
  }
  const int64_t chunks = cap / kSortChunk;
  if ((rc = grow(ctx, ctx->sort_status, (int64_t)kMaxPasses * chunks * kRadix)) != GS_OK) return rc;
  ctx->cap_sort_chunks = chunks;
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

int launch_binning(gs_ctx* ctx, cudaStream_t s) {
  const int64_t tiles = (int64_t)ctx->cam.tiles_x * ctx->cam.tiles_y;
  GS_PROF(2, s);
  GS_CUDA(cudaMemsetAsync(ctx->ranges, 0, (size_t)tiles * sizeof(uint2), s));
  if (ctx->N == 0) {
    GS_CUDA(cudaMemsetAsync(ctx->counts, 0, sizeof(Counts), s));
    tile_order_kernel<<<1, 1024, 0, s>>>((int)tiles, ctx->ranges, ctx->tile_order);
    GS_LAUNCH_CHECK("tile_order_kernel");
    return GS_OK;
  }
  const bool same_shape = ctx->calibrated && ctx->cal_N == ctx->N && ctx->cal_W == ctx->cam.W && ctx->cal_H == ctx->cam.H;
  int rc;
  if (!same_shape) {
    // calibration: run the scan once (emitting nothing if the capacity is short), read the instance count, size the
    // buffers, and run it again if it overflowed.  This is the only synchronising path of the iteration.
    if ((rc = run_scan_dup(ctx, s)) != GS_OK) return rc;
    GS_CUDA(cudaStreamSynchronize(s));
    const int64_t I = ctx->mailbox->n_instances;
    if (I > ctx->cap_I) {
      if ((rc = ensure_instance_capacity(ctx, I)) != GS_OK) return rc;
      if ((rc = run_scan_dup(ctx, s)) != GS_OK) return rc;
    }
    ctx->calibrated = true;
    ctx->cal_N = ctx->N; ctx->cal_W = ctx->cam.W; ctx->cal_H = ctx->cam.H;
  } else {
    // asynchronous path: act on what the last finished iteration reported (no synchronisation): an overflow is
    // reported to the caller (after growing), a near-full buffer is grown ahead of time
    if (handle_overflow(ctx)) return fail(ctx, GS_E_OVERFLOW, "tile-instance capacity exceeded in an earlier iteration; scratch has grown, re-issue");
    const Counts mb = read_mailbox(ctx);
    if ((int64_t)mb.n_instances + (int64_t)mb.n_instances / 8 > ctx->cap_I)
      if ((rc = ensure_instance_capacity(ctx, (int64_t)mb.n_instances + (int64_t)mb.n_instances / 4)) != GS_OK) return rc;
    if ((rc = run_scan_dup(ctx, s)) != GS_OK) return rc;
  }
  GS_PROF(3, s);
  // radix sort plan: 4 depth digits + ceil(tile_bits / 8) tile digits
  SortPlan plan;
  plan.passes = 0;
  for (int b = 0; b < 32; b += kRadixBits) plan.shift[plan.passes++] = b;
  int tile_bits = 0;
  while ((1ll << tile_bits) < tiles) ++tile_bits;
  for (int b = 0; b < tile_bits; b += kRadixBits) plan.shift[plan.passes++] = 32 + b;
  const int64_t chunks = ctx->cap_sort_chunks;
  GS_CUDA(cudaMemsetAsync(ctx->sort_hist, 0, (size_t)kMaxPasses * kRadix * sizeof(uint32_t), s));
  GS_CUDA(cudaMemsetAsync(ctx->sort_status, 0, (size_t)plan.passes * chunks * kRadix * sizeof(uint32_t), s));
  sort_hist_kernel<<<(unsigned)chunks, kSortThreads, 0, s>>>(ctx->keys[0], ctx->counts, plan, ctx->sort_hist);
  GS_LAUNCH_CHECK("sort_hist_kernel");
  int cur = 0;
  for (int p = 0; p < plan.passes; ++p) {
    sort_pass_kernel<<<(unsigned)chunks, kSortThreads, 0, s>>>(
        ctx->keys[cur], ctx->vals[cur], ctx->keys[cur ^ 1], ctx->vals[cur ^ 1], ctx->counts, plan.shift[p],
        ctx->sort_hist + p * kRadix, ctx->sort_status + (size_t)p * chunks * kRadix, ctx->sort_ticket + p);
    GS_LAUNCH_CHECK("sort_pass_kernel");
    cur ^= 1;
  }
  ctx->sorted_buf = cur;
  GS_PROF(4, s);
  const int threads = 256;
  tile_ranges_kernel<<<(unsigned)div_up(ctx->cap_I, threads), threads, 0, s>>>(ctx->keys[cur], ctx->counts, ctx->ranges);
  GS_LAUNCH_CHECK("tile_ranges_kernel");
  tile_order_kernel<<<1, 1024, 0, s>>>((int)tiles, ctx->ranges, ctx->tile_order);
  GS_LAUNCH_CHECK("tile_order_kernel");
  GS_PROF(5, s);
  return GS_OK;
}

}  // namespace gs
