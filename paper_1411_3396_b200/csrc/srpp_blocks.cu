// srpp_blocks.cu -- block decomposition of the node volume with the x2 adaptive refinement rule (SURVEY.md 8(f)
// item 2; Sec. 2.1 "HACC: Load-Balancing on the GPU").
//
// The paper's scheme, per short-range force timestep: "1) Each node partitions itself into overlapping data blocks,
// 2) evolves the blocks independently, and 3) reconciles the alive particles, whereby removing the unnecessary
// duplicated passive ones"; the blocks' "x-axis is equally partitioned in PM grid units" and a block
// whose "timing is more than a factor of two larger than the average" is "divided a factor of two finer"
// (PAPER.md:75-77).  On one GPU (BASELINE.json: no sharding) the blocks are evaluated one after the other; what is
// built here is exactly the per-block machinery and the refinement policy:
//   * a block = active x-range [x0, x1) (integer PM grid units) + a passive shell of >= rc on both sides; its
//     particles are EXTRACTED into their own arrays (k_block_count / k_block_extract, stable order) in a block-local
//     frame whose origin is an integer, so the shift is exact in fp32 (except for the shell that wraps through the
//     periodic face at x = L, where x + K rounds -- those particles are passive sources);
//   * the block is an independent problem: its own srpp context (open x faces, the parent's y and z), its own
//     chaining mesh, srpp_set_boundary(active box), srpp_accel -- "one can picture each node as a separate HACC
//     simulation";
//   * reconcile: the accelerations of the particles with x0 <= x < x1 go back to the caller's array
//     (k_block_reconcile); the duplicated passive copies are dropped;
//   * every block is timed with CUDA events; after the pass the plan for the NEXT call is refined: a block slower than
//     twice the mean block time is split in two halves (never below 1 grid unit, at most kMaxBlocks blocks).
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "srpp_internal.cuh"

namespace srpp {

constexpr int kExtractTile = 1024;

// block-local x of a particle, or a negative value if it is not in [o, o + len) (periodic in x with length L)
__device__ __forceinline__ float block_local_x(float x, float o, float len, float L) {
  float xl = x - o;                          // exact: o is an integer below x's magnitude range (see header)
  if (xl >= 0.f && xl < len) return xl;
  xl = (x - L) - o;                          // image one box length below: both subtractions exact
  if (xl >= 0.f && xl < len) return xl;
  xl = x + (L - o);                          // image one box length above (rounds: these are passive sources)
  if (xl >= 0.f && xl < len) return xl;
  return -1.f;
}

__global__ void __launch_bounds__(kExtractTile) k_block_count(const float4* __restrict__ pos, int64_t n, float o, float len,
                                                               float L, unsigned long long* __restrict__ tile_count) {
  const int64_t i = (int64_t)blockIdx.x * kExtractTile + threadIdx.x;
  const bool in = i < n && block_local_x(__ldg(&pos[i].x), o, len, L) >= 0.f;
  const int c = __syncthreads_count(in);
  if (threadIdx.x == 0) tile_count[blockIdx.x] = (unsigned long long)c;
}

// stable compaction: tile_prefix = exclusive scan of tile_count
__global__ void __launch_bounds__(kExtractTile) k_block_extract(const float4* __restrict__ pos, int64_t n, float o, float len,
                                                                 float L, const unsigned long long* __restrict__ tile_prefix,
                                                                 float4* __restrict__ bpos, uint32_t* __restrict__ bidx) {
  __shared__ uint32_t wsum[32];
  const int64_t i = (int64_t)blockIdx.x * kExtractTile + threadIdx.x;
  float4 p = make_float4(0.f, 0.f, 0.f, 0.f);
  float xl = -1.f;
  if (i < n) { p = __ldg(&pos[i]); xl = block_local_x(p.x, o, len, L); }
  const bool in = xl >= 0.f;
  const uint32_t bal = __ballot_sync(0xffffffffu, in);
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  if (lane == 0) wsum[w] = __popc(bal);
  __syncthreads();
  if (w == 0) {
    uint32_t v = wsum[lane], x = v;
#pragma unroll
    for (int s = 1; s < 32; s <<= 1) { const uint32_t y = __shfl_up_sync(0xffffffffu, x, s); if (lane >= s) x += y; }
    wsum[lane] = x - v;
  }
  __syncthreads();
  if (in) {
    const size_t dst = (size_t)tile_prefix[blockIdx.x] + wsum[w] + __popc(bal & ((1u << lane) - 1u));
    p.x = xl;
    bpos[dst] = p;
    bidx[dst] = (uint32_t)i;
  }
}

// reconcile: the active particles' accelerations go back to the caller's order; passive copies are dropped
__global__ void __launch_bounds__(256) k_block_reconcile(const float4* __restrict__ pos, const uint32_t* __restrict__ bidx,
                                                          const float4* __restrict__ bacc, int64_t nb, float x0, float x1,
                                                          float4* __restrict__ acc, unsigned long long* __restrict__ n_active) {
  const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  bool act = false;
  if (j < nb) {
    const uint32_t i = bidx[j];
    const float x = __ldg(&pos[i].x);          // the test is made on the caller's coordinate: every particle is active in exactly one block
    act = x >= x0 && x < x1;
    if (act) acc[i] = bacc[j];
  }
  const uint32_t bal = __ballot_sync(0xffffffffu, act);
  if ((threadIdx.x & 31) == 0 && bal) atomicAdd(n_active, (unsigned long long)__popc(bal));
}

}  // namespace srpp

using namespace srpp;

struct BlockPlan {
  int32_t count;
  float x0[SRPP_MAX_BLOCKS], x1[SRPP_MAX_BLOCKS];
  int32_t level[SRPP_MAX_BLOCKS];
  srpp_block_info last[SRPP_MAX_BLOCKS];
  int32_t last_count;
};

namespace srpp { void free_block_plan(srpp_ctx* c); }
static BlockPlan* plan_of(srpp_ctx* c) { return (BlockPlan*)c->block_plan; }

static size_t align256(size_t x) { return (x + 255) / 256 * 256; }

// sub-geometry of a block of active length `len_active` (grid units): frame [o, o + lb), cells of edge >= max(rc, parent cell)
static void block_geometry(const srpp_params& P, float x0, float x1, float* o, float* lb, int32_t* ncx) {
  const float pad = P.rcut;
  *o = floorf(x0 - pad);
  const float e = ceilf(x1 + pad);
  *lb = e - *o;
  const float wcell = fmaxf(P.rcut, P.box[0] / (float)P.ncell[0]);
  int32_t k = (int32_t)floorf(*lb / wcell);
  if (k < 3) k = 3;
  while (k > 3 && (double)*lb / k < (double)P.rcut) --k;
  if ((double)*lb / k < (double)P.rcut) *lb = ceilf(3.f * P.rcut);   // a narrow block: widen the upper shell to 3 cells of edge rc
  *ncx = k;
}

void srpp::free_block_plan(srpp_ctx* c) {
  delete (BlockPlan*)c->block_plan;
  c->block_plan = nullptr;
}

extern "C" {

int32_t srpp_blocks_workspace_bytes(const srpp_params* params, int64_t n, size_t* bytes_host) {
  if (!params || !bytes_host || n < 0 || n >= ((int64_t)1 << 31)) return SRPP_ERR_INVALID_ARG;
  // a block's frame is shorter than the box and its cells are no smaller than the parent's, so it never has more
  // cells than the parent mesh: the parent's workspace size bounds every block's
  size_t inner = 0;
  const int32_t rc = srpp_workspace_bytes(params, n, &inner);
  if (rc != SRPP_OK) return rc;
  const size_t nn = (size_t)(n > 0 ? n : 1);
  *bytes_host = align256(inner) + align256(16 * nn) * 2 + align256(4 * nn) + align256(8 * (nn / kExtractTile + 2)) * 2 + 256;
  return SRPP_OK;
}

int32_t srpp_blocks_init(srpp_ctx* c, int32_t nblocks) {
  if (!c || nblocks < 1 || nblocks > SRPP_MAX_BLOCKS) return SRPP_ERR_INVALID_ARG;
  const float L = c->params.box[0];
  if (L != floorf(L) || (float)nblocks > L) return SRPP_ERR_GEOMETRY;      // boundaries are integer PM grid units
  if (!c->block_plan) {
    c->block_plan = new (std::nothrow) BlockPlan();
    if (!c->block_plan) return SRPP_ERR_INVALID_ARG;
  }
  BlockPlan* bp = plan_of(c);
  memset(bp, 0, sizeof(*bp));
  bp->count = nblocks;
  for (int32_t b = 0; b < nblocks; ++b) {          // "the x-axis is equally partitioned in PM grid units"
    bp->x0[b] = floorf((float)((double)L * b / nblocks + 0.5));
    bp->x1[b] = b == nblocks - 1 ? L : floorf((float)((double)L * (b + 1) / nblocks + 0.5));
    bp->level[b] = 0;
  }
  return SRPP_OK;
}

int32_t srpp_get_blocks(const srpp_ctx* c, srpp_block_info* out_host, int32_t capacity, int32_t* count_host) {
  if (!c || !count_host || capacity < 0 || (capacity > 0 && !out_host)) return SRPP_ERR_INVALID_ARG;
  const BlockPlan* bp = (const BlockPlan*)c->block_plan;
  if (!bp) return SRPP_ERR_STATE;
  *count_host = bp->last_count;
  for (int32_t b = 0; b < bp->last_count && b < capacity; ++b) out_host[b] = bp->last[b];
  return SRPP_OK;
}

int32_t srpp_accel_blocks(srpp_ctx* c, const float* pos_mass, int64_t n, float* acc, void* workspace, size_t workspace_bytes) {
  if (!c || n < 0 || n >= ((int64_t)1 << 31) || (n > 0 && (!pos_mass || !acc)) || !workspace ||
      ((uintptr_t)pos_mass & 15u) || ((uintptr_t)acc & 15u))
    return SRPP_ERR_INVALID_ARG;
  BlockPlan* bp = plan_of(c);
  if (!bp || bp->count < 1) return SRPP_ERR_STATE;
  size_t need = 0;
  int32_t rc = srpp_blocks_workspace_bytes(&c->params, n, &need);
  if (rc != SRPP_OK) return rc;
  if (((uintptr_t)workspace & 255u) || workspace_bytes < need) return SRPP_ERR_WORKSPACE;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return SRPP_ERR_CUDA;
  if (dev != c->device) return SRPP_ERR_STATE;
  cudaStream_t st = c->stream;
  const srpp_params& P = c->params;
  const float L = P.box[0];
  const size_t nn = (size_t)(n > 0 ? n : 1);

  // carve: [inner workspace | block positions | block accelerations | block indices | tile counts | scan scratch | counters]
  char* w = (char*)workspace;
  size_t inner = 0;
  srpp_workspace_bytes(&P, n, &inner);
  char* w_inner = w; w += align256(inner);
  float4* bpos = (float4*)w; w += align256(16 * nn);
  float4* bacc = (float4*)w; w += align256(16 * nn);
  uint32_t* bidx = (uint32_t*)w; w += align256(4 * nn);
  unsigned long long* tcount = (unsigned long long*)w; w += align256(8 * (nn / kExtractTile + 2));
  unsigned long long* ttmp = (unsigned long long*)w; w += align256(8 * (nn / kExtractTile + 2));
  unsigned long long* counters = (unsigned long long*)w;      // [0] block size, [1] active count

  cudaEvent_t ev0 = nullptr, ev1 = nullptr;
  cudaError_t e = cudaEventCreate(&ev0);
  if (e == cudaSuccess) e = cudaEventCreate(&ev1);
  if (e != cudaSuccess) { if (ev0) cudaEventDestroy(ev0); return SRPP_ERR_CUDA; }
  auto fail = [&](int32_t code) { cudaEventDestroy(ev0); cudaEventDestroy(ev1); return code; };

  if (n > 0 && cudaMemsetAsync(acc, 0, 16 * (size_t)n, st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
  const int ntile = (int)((n + kExtractTile - 1) / kExtractTile);
  bp->last_count = 0;
  for (int32_t b = 0; b < bp->count; ++b) {
    const float x0 = bp->x0[b], x1 = bp->x1[b];
    srpp_block_info info;
    memset(&info, 0, sizeof(info));
    info.x0 = x0; info.x1 = x1; info.level = bp->level[b];
    if (cudaEventRecord(ev0, st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
    if (n > 0) {
      srpp_params sub = P;
      float o = 0.f, lb = L;
      int32_t periodic[3] = {1, c->geo.periodic[1], c->geo.periodic[2]};
      float alo[3] = {0.f, 0.f, 0.f}, ahi[3] = {L, P.box[1], P.box[2]};
      const float l_img = c->geo.periodic[0] ? L : 4.f * L;      // an open parent x axis has no images across its faces
      const bool whole = bp->count == 1 || (x1 - x0) + 2.f * P.rcut + 2.f >= L;   // the block and its shell cover the box:
      if (whole) {                                                                 // evaluate the periodic box as it is
        periodic[0] = c->geo.periodic[0];
        alo[0] = x0; ahi[0] = x1;
      } else {
        int32_t ncx = 3;
        block_geometry(P, x0, x1, &o, &lb, &ncx);
        sub.box[0] = lb;
        sub.ncell[0] = ncx;
        periodic[0] = 0;                                                           // open faces: the shell replaces the wrap
        alo[0] = x0 - o; ahi[0] = x1 - o;
      }
      // 1) partition: extract the block (active range + passive shell), stable order, block-local frame
      k_block_count<<<ntile, kExtractTile, 0, st>>>((const float4*)pos_mass, n, o, lb, whole ? 4.f * L : l_img, tcount);
      if ((e = launch_scan_u64(st, tcount, ntile, ttmp, &counters[0], &counters[2])) != cudaSuccess) return fail(SRPP_ERR_CUDA);
      k_block_extract<<<ntile, kExtractTile, 0, st>>>((const float4*)pos_mass, n, o, lb, whole ? 4.f * L : l_img, tcount, bpos, bidx);
      unsigned long long nb_host = 0;
      if (cudaMemsetAsync(&counters[1], 0, 8, st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
      if (cudaMemcpyAsync(&nb_host, &counters[0], 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
      if (cudaStreamSynchronize(st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
      c->launches += 5;
      const int64_t nb = (int64_t)nb_host;
      info.n_total = nb;
      if (nb > 0) {
        // 2) evolve the block independently: its own context, mesh and force evaluation
        srpp_ctx* bc = nullptr;
        if ((rc = srpp_create(&bc, &sub, w_inner, align256(inner), st)) != SRPP_OK) return fail(rc);
        rc = srpp_set_boundary(bc, periodic, alo, ahi);
        if (rc == SRPP_OK) rc = srpp_build_mesh(bc, (const float*)bpos, nb);
        if (rc == SRPP_OK) rc = srpp_accel(bc, (float*)bacc);
        srpp_stats stt;
        memset(&stt, 0, sizeof(stt));
        if (rc == SRPP_OK) rc = srpp_get_stats(bc, &stt);
        if (rc == SRPP_ERR_CUDA) snprintf(c->cuda_err, sizeof(c->cuda_err), "%s", srpp_last_cuda_error(bc));
        c->launches += stt.kernel_launches;
        srpp_destroy(bc);
        if (rc != SRPP_OK) return fail(rc);
        info.candidate_pairs = stt.candidate_pairs;
        // 3) reconcile: active particles back to the caller's array
        k_block_reconcile<<<(int)((nb + 255) / 256), 256, 0, st>>>((const float4*)pos_mass, bidx, bacc, nb, x0, x1, (float4*)acc, &counters[1]);
        c->launches += 1;
      }
    }
    if (cudaEventRecord(ev1, st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
    unsigned long long nact = 0;
    if (n > 0 && cudaMemcpyAsync(&nact, &counters[1], 8, cudaMemcpyDeviceToHost, st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
    if (cudaStreamSynchronize(st) != cudaSuccess) return fail(SRPP_ERR_CUDA);
    info.n_active = (int64_t)nact;
    cudaEventElapsedTime(&info.ms, ev0, ev1);
    bp->last[bp->last_count++] = info;
  }
  cudaEventDestroy(ev0);
  cudaEventDestroy(ev1);

  // the x2 rule for the NEXT call: a block slower than twice the mean is divided a factor of two finer
  double mean = 0.0;
  for (int32_t b = 0; b < bp->last_count; ++b) mean += bp->last[b].ms;
  mean /= std::max(1, bp->last_count);
  BlockPlan next = *bp;
  next.count = 0;
  for (int32_t b = 0; b < bp->count; ++b) {
    const float x0 = bp->x0[b], x1 = bp->x1[b];
    const int32_t remaining = bp->count - b - 1;
    const bool split = bp->last[b].ms > 2.0 * mean && x1 - x0 >= 2.f && next.count + 2 + remaining <= SRPP_MAX_BLOCKS;
    if (split) {
      const float xm = floorf(0.5f * (x0 + x1));
      next.x0[next.count] = x0; next.x1[next.count] = xm; next.level[next.count++] = bp->level[b] + 1;
      next.x0[next.count] = xm; next.x1[next.count] = x1; next.level[next.count++] = bp->level[b] + 1;
    } else {
      next.x0[next.count] = x0; next.x1[next.count] = x1; next.level[next.count++] = bp->level[b];
    }
  }
  bp->count = next.count;
  memcpy(bp->x0, next.x0, sizeof(bp->x0));
  memcpy(bp->x1, next.x1, sizeof(bp->x1));
  memcpy(bp->level, next.level, sizeof(bp->level));
  return SRPP_OK;
}

}  // extern "C"
