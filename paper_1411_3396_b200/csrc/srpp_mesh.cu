// srpp_mesh.cu -- chaining-mesh binning (steps A1-A4 of SURVEY.md 8(a)) for sm_100a.
//
// The mesh is a STABLE counting sort of the particles by linear cell id (readings R10-R12):
//   A1  cell id per particle, fp32:  c = min((int)floorf(x * inv), ncell-1), inv = (float)ncell/box
//   A2-A4 histogram / exclusive scan / stable scatter.  To stay deterministic and HBM-friendly for up to
//        2^24 cells and cells holding millions of particles, the counting sort is applied digit-wise
//        (8-bit LSD digits of the cell id): each pass is a per-block digit histogram (upsweep), an exclusive
//        scan over (digit, block), and a stable scatter (downsweep) whose in-block ranks come from
//        warp match + per-warp digit counters.  No atomics decide an output position, so perm is
//        bit-exact reproducible and equals the oracle's stable counting sort.
//   cell_start = run boundaries of the sorted ids (= exclusive prefix sum of the cell histogram);
//   sorted[k]  = pos_mass[perm[k]] gathered in the same pass.
// Paper context: PAPER.md:63/65 (direct PP short-range solver inside the hand-over radius); the chaining
// mesh itself is named by BASELINE.json north_star.
#include <algorithm>

#include "srpp_internal.cuh"

namespace srpp {

// ------------------------------------------------------------------------------- A1: cell ids --
__global__ void __launch_bounds__(256) k_cell_ids(const float4* __restrict__ pos_mass, int64_t n, Geometry g,
                                                   uint32_t* __restrict__ cid, DevFlags* flags) {
  const float m0 = n > 0 ? __ldg(&pos_mass[0].w) : 0.f;
  uint32_t bad = 0, mdiff = 0;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) {
    const float4 p = __ldg(&pos_mass[i]);
    const bool ok = (p.x >= 0.f) && (p.x < g.box[0]) && (p.y >= 0.f) && (p.y < g.box[1]) && (p.z >= 0.f) &&
                    (p.z < g.box[2]);
    // one IEEE multiply per axis (never contracted: there is nothing to fuse with), floor, clamp (R10)
    int cx = (int)floorf(__fmul_rn(p.x, g.inv_cell[0]));
    int cy = (int)floorf(__fmul_rn(p.y, g.inv_cell[1]));
    int cz = (int)floorf(__fmul_rn(p.z, g.inv_cell[2]));
    cx = min(cx, g.ncell[0] - 1);
    cy = min(cy, g.ncell[1] - 1);
    cz = min(cz, g.ncell[2] - 1);
    uint32_t id = ok ? (uint32_t)cx + (uint32_t)g.ncell[0] * ((uint32_t)cy + (uint32_t)g.ncell[1] * (uint32_t)cz) : 0u;
    cid[i] = id;
    bad |= ok ? 0u : 1u;
    mdiff |= (p.w != m0) ? 1u : 0u;   // NaN mass counts as different
  }
  if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(&flags->domain_error, 1u);
  if (__any_sync(0xffffffffu, mdiff) && (threadIdx.x & 31) == 0) atomicOr(&flags->mass_nonuniform, 1u);
}

// ------------------------------------------------------------------- A2: per-block digit histogram --
__global__ void __launch_bounds__(kSortThreads) k_radix_upsweep(const uint32_t* __restrict__ keys, int64_t n, int shift,
                                                                 uint32_t* __restrict__ hist, int nblocks,
                                                                 int tiles_per_block) {
  __shared__ uint32_t h[kRadix];
  h[threadIdx.x] = 0;
  __syncthreads();
  const int64_t beg = (int64_t)blockIdx.x * tiles_per_block * kSortTile;
  const int64_t end = min(n, beg + (int64_t)tiles_per_block * kSortTile);
  for (int64_t i = beg + threadIdx.x; i < end; i += kSortThreads) {
    const uint32_t d = (__ldg(&keys[i]) >> shift) & (kRadix - 1);
    // warp-aggregate equal digits so a heavy cell does not serialise on one shared-memory word
    const uint32_t active = __activemask();
    const uint32_t peers = __match_any_sync(active, d);
    if ((threadIdx.x & 31) == (__ffs(peers) - 1)) atomicAdd(&h[d], (uint32_t)__popc(peers));
  }
  __syncthreads();
  hist[(size_t)threadIdx.x * nblocks + blockIdx.x] = h[threadIdx.x];
}

// ------------------------------------------------- A3: exclusive scan over (digit-major, block-minor) --
__global__ void __launch_bounds__(1024) k_radix_scan(uint32_t* __restrict__ hist, int total) {
  __shared__ uint32_t warp_sums[32];
  __shared__ uint32_t carry;
  if (threadIdx.x == 0) carry = 0;
  __syncthreads();
  const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
  for (int base = 0; base < total; base += 1024) {
    const int i = base + threadIdx.x;
    const uint32_t v = i < total ? hist[i] : 0u;
    uint32_t x = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t y = __shfl_up_sync(0xffffffffu, x, o);
      if (lane >= o) x += y;
    }
    if (lane == 31) warp_sums[wid] = x;
    __syncthreads();
    if (wid == 0) {
      uint32_t w = warp_sums[lane];
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t y = __shfl_up_sync(0xffffffffu, w, o);
        if (lane >= o) w += y;
      }
      warp_sums[lane] = w;  // inclusive
    }
    __syncthreads();
    const uint32_t before = carry + (wid ? warp_sums[wid - 1] : 0u) + (x - v);
    if (i < total) hist[i] = before;
    __syncthreads();
    if (threadIdx.x == 1023) carry = before + v;
    __syncthreads();
  }
}

// ---------------------------------------------------------------------- A4: stable scatter of a digit --
// Warp w of the CTA owns keys [tile + 256w, tile + 256w + 256) and walks them in 8 steps of 32 consecutive
// keys, so (block, tile, warp, step, lane) order == original order; ranks are assigned in that order.
template <bool kIdentityVals>
__global__ void __launch_bounds__(kSortThreads) k_radix_downsweep(const uint32_t* __restrict__ keys_in,
                                                                   const uint32_t* __restrict__ vals_in,
                                                                   uint32_t* __restrict__ keys_out,
                                                                   uint32_t* __restrict__ vals_out, int64_t n, int shift,
                                                                   const uint32_t* __restrict__ hist, int nblocks,
                                                                   int tiles_per_block) {
  __shared__ uint32_t base[kRadix];
  __shared__ uint32_t wc[kSortThreads / 32][kRadix];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const uint32_t lt_mask = (1u << lane) - 1u;
  base[threadIdx.x] = hist[(size_t)threadIdx.x * nblocks + blockIdx.x];
  const int64_t beg = (int64_t)blockIdx.x * tiles_per_block * kSortTile;
  const int64_t end = min(n, beg + (int64_t)tiles_per_block * kSortTile);
  for (int64_t tile = beg; tile < end; tile += kSortTile) {
#pragma unroll
    for (int r = 0; r < kSortThreads / 32; ++r) wc[r][threadIdx.x] = 0;
    __syncthreads();
    uint32_t key[kSortKeysPerThread], val[kSortKeysPerThread], rank[kSortKeysPerThread];
    const int64_t wbase = tile + (int64_t)w * (32 * kSortKeysPerThread);
#pragma unroll
    for (int s = 0; s < kSortKeysPerThread; ++s) {
      const int64_t i = wbase + s * 32 + lane;
      const bool valid = i < end;
      key[s] = valid ? __ldg(&keys_in[i]) : 0u;
      val[s] = kIdentityVals ? (uint32_t)i : (valid ? __ldg(&vals_in[i]) : 0u);
    }
#pragma unroll
    for (int s = 0; s < kSortKeysPerThread; ++s) {
      const int64_t i = wbase + s * 32 + lane;
      const bool valid = i < end;
      const uint32_t d = (key[s] >> shift) & (kRadix - 1);
      // invalid lanes get a unique pseudo-digit so they never join a peer group
      const uint32_t peers = __match_any_sync(0xffffffffu, valid ? d : (0x10000u + (uint32_t)lane));
      const uint32_t prev = valid ? wc[w][d] : 0u;
      rank[s] = prev + (uint32_t)__popc(peers & lt_mask);
      __syncwarp();
      if (valid && lane == (__ffs(peers) - 1)) wc[w][d] = prev + (uint32_t)__popc(peers);
      __syncwarp();
    }
    __syncthreads();
    {  // exclusive prefix over the 8 warps for digit == threadIdx.x, on top of the running global base
      uint32_t run = base[threadIdx.x];
#pragma unroll
      for (int r = 0; r < kSortThreads / 32; ++r) {
        const uint32_t c = wc[r][threadIdx.x];
        wc[r][threadIdx.x] = run;
        run += c;
      }
      base[threadIdx.x] = run;
    }
    __syncthreads();
#pragma unroll
    for (int s = 0; s < kSortKeysPerThread; ++s) {
      const int64_t i = wbase + s * 32 + lane;
      if (i < end) {
        const uint32_t d = (key[s] >> shift) & (kRadix - 1);
        const uint32_t dst = wc[w][d] + rank[s];
        keys_out[dst] = key[s];
        vals_out[dst] = val[s];
      }
    }
    __syncthreads();
  }
}

// --------------------------------------------- cell_start from run boundaries + gather of sorted[] --
__global__ void __launch_bounds__(256) k_finalize_mesh(const uint32_t* __restrict__ sorted_keys,
                                                        const uint32_t* __restrict__ perm,
                                                        const float4* __restrict__ pos_mass, int64_t n, int32_t ncells,
                                                        uint32_t* __restrict__ cell_start, float4* __restrict__ sorted) {
  for (int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (int64_t)gridDim.x * blockDim.x) {
    const uint32_t key = __ldg(&sorted_keys[k]);
    const int64_t prev = k > 0 ? (int64_t)__ldg(&sorted_keys[k - 1]) : -1;
    // cells (prev, key] start at k: the first is `key` itself, the rest are empty cells before it
    for (int64_t c = prev + 1; c <= (int64_t)key; ++c) cell_start[c] = (uint32_t)k;
    if (k == n - 1)
      for (int64_t c = (int64_t)key + 1; c <= (int64_t)ncells; ++c) cell_start[c] = (uint32_t)n;
    sorted[k] = __ldg(&pos_mass[__ldg(&perm[k])]);
  }
}

cudaError_t launch_build_mesh(srpp_ctx* c, const float4* pos_mass, int64_t n) {
  cudaStream_t st = c->stream;
  cudaError_t e;
  if ((e = cudaMemsetAsync(c->flags, 0, sizeof(DevFlags), st)) != cudaSuccess) return e;
  const int32_t ncells = c->geo.ncells;
  if (n == 0) {
    c->perm = c->vals[0];
    c->sorted_keys = c->keys[0];
    return cudaMemsetAsync(c->cell_start, 0, sizeof(uint32_t) * ((size_t)ncells + 1), st);
  }
  if (c->timing) cudaEventRecord(c->ev[kEvMesh0], st);
  const int grid_ew = (int)std::min<int64_t>((n + 255) / 256, (int64_t)c->num_sms * 16);
  k_cell_ids<<<grid_ew, 256, 0, st>>>(pos_mass, n, c->geo, c->keys[0], c->flags);

  const int64_t tiles = (n + kSortTile - 1) / kSortTile;
  int blocks = (int)std::min<int64_t>(tiles, (int64_t)c->num_sms * kSortBlocksPerSM);
  const int tpb = (int)((tiles + blocks - 1) / blocks);
  blocks = (int)((tiles + tpb - 1) / tpb);
  c->sort_blocks = blocks;
  for (int p = 0; p < c->sort_passes; ++p) {
    const uint32_t* kin = c->keys[p & 1];
    const uint32_t* vin = c->vals[p & 1];
    uint32_t* kout = c->keys[(p + 1) & 1];
    uint32_t* vout = c->vals[(p + 1) & 1];
    const int shift = p * kRadixBits;
    k_radix_upsweep<<<blocks, kSortThreads, 0, st>>>(kin, n, shift, c->hist, blocks, tpb);
    k_radix_scan<<<1, 1024, 0, st>>>(c->hist, kRadix * blocks);
    if (p == 0)
      k_radix_downsweep<true><<<blocks, kSortThreads, 0, st>>>(kin, nullptr, kout, vout, n, shift, c->hist, blocks, tpb);
    else
      k_radix_downsweep<false><<<blocks, kSortThreads, 0, st>>>(kin, vin, kout, vout, n, shift, c->hist, blocks, tpb);
  }
  c->perm = c->vals[c->sort_passes & 1];
  c->sorted_keys = c->keys[c->sort_passes & 1];
  k_finalize_mesh<<<grid_ew, 256, 0, st>>>(c->sorted_keys, c->perm, pos_mass, n, ncells, c->cell_start, c->sorted);
  c->launches += 2 + 3 * (uint64_t)c->sort_passes;
  if (c->timing) { cudaEventRecord(c->ev[kEvMesh1], st); c->ev_mesh_valid = true; }
  return cudaGetLastError();
}

}  // namespace srpp
