// srpp_mbp.cu -- most-bound-particle halo centre finder for sm_100a.
//
//   phi_i = - sum_{j in halo, j != i} m_j / sqrt(|x_j - x_i|^2 + eps^2),   centre = argmin_i phi_i  (lowest index on ties)
//
// The paper builds this from Thrust scan/transform/reduce on Titan's K20X; here it is the second O(n^2) workload on
// the pair-tile machinery of the force kernel:
//   * work item = (halo h, tile of <= 128 members as targets, chunk of <= 1024 members as sources); all items of all
//     halos form one index space (exclusive prefix over halos, computed on the device from halo_start) and autonomous
//     warps pull items from one atomic counter, so a 4-million-particle halo spreads over the whole chip while 10^5
//     small halos fill it just as well (the paper's load imbalance across halos);
//   * targets in registers as packed pairs, sources staged per warp as float4 (x, y, z, m) relative to the halo's first
//     member, one LDS.128 per source, packed FADD2/FFMA2 arithmetic, one MUFU.RSQ per pair;
//   * the self pair is included in the stream (d = 0 exactly, term m_i * rsqrt(eps^2)) and removed afterwards;
//   * <= 1024 fp32 terms per item, folded into fp64 with red.global.add.f64; a second kernel negates, removes the self
//     term and reduces (phi, index) per halo.
#include <algorithm>

#include "srpp_internal.cuh"

namespace srpp {

constexpr int kMbpTargets = 128;      // targets per item: 32 lanes x 2 packed pairs
constexpr int kMbpChunk = 1024;       // sources per item

__device__ __forceinline__ float mbp_rsqrt(float x) {
  float y;
  asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}

struct __align__(16) MbpScratch {
  float4 src[kSrcTile];
};

__global__ void __launch_bounds__(kForceThreads, 2)
k_mbp_phi(const float4* __restrict__ pos_mass, const long long* __restrict__ halo_start,
          const unsigned long long* __restrict__ item_prefix, int nhalo, float eps2, unsigned long long* counter,
          double* __restrict__ phi64) {
  __shared__ MbpScratch scratch[kForceWarps];
  const int lane = threadIdx.x & 31;
  MbpScratch& ws = scratch[threadIdx.x >> 5];
  const unsigned long long total = __ldg(&item_prefix[nhalo]);
  const float2 e2 = make_float2(eps2, eps2);
  for (;;) {
    unsigned long long idx = 0;
    if (lane == 0) idx = atomicAdd(counter, 1ull);
    idx = __shfl_sync(0xffffffffu, idx, 0);
    if (idx >= total) break;
    // 32-ary search: largest h with item_prefix[h] <= idx
    int lo = 0, hi = nhalo;
    while (hi - lo > 1) {
      const int step = (hi - lo + 31) / 32;
      const int probe = lo + lane * step;
      const bool le = (probe < hi) && (__ldg(&item_prefix[probe]) <= idx);
      const int k = __popc(__ballot_sync(0xffffffffu, le));
      const int nlo = lo + (k - 1) * step;
      hi = min(hi, nlo + step);
      lo = nlo;
    }
    const int h = lo;
    const long long hb = __ldg(&halo_start[h]), he = __ldg(&halo_start[h + 1]);
    const unsigned long long local = idx - __ldg(&item_prefix[h]);
    const unsigned long long ntile = (unsigned long long)((he - hb + kMbpTargets - 1) / kMbpTargets);
    const long long tb = hb + (long long)(local % ntile) * kMbpTargets, te = min(he, tb + kMbpTargets);
    const long long p0 = hb + (long long)(local / ntile) * kMbpChunk, p1 = min(he, p0 + kMbpChunk);
    const float4 ref = __ldg(&pos_mass[hb]);

    float2 ntx[2], nty[2], ntz[2], phi[2];
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      const long long k0 = tb + t * 64 + lane, k1 = k0 + 32;
      float4 a = make_float4(ref.x, ref.y, ref.z, 0.f), b = a;
      if (k0 < te) a = __ldg(&pos_mass[k0]);
      if (k1 < te) b = __ldg(&pos_mass[k1]);
      ntx[t] = make_float2(-(a.x - ref.x), -(b.x - ref.x));
      nty[t] = make_float2(-(a.y - ref.y), -(b.y - ref.y));
      ntz[t] = make_float2(-(a.z - ref.z), -(b.z - ref.z));
      phi[t] = make_float2(0.f, 0.f);
    }
    for (long long tile = p0; tile < p1; tile += kSrcTile) {
      __syncwarp();
#pragma unroll
      for (int j = 0; j < kSrcTile / 32; ++j) {
        const long long p = tile + j * 32 + lane;
        float4 sv = make_float4(0.f, 0.f, 0.f, 0.f);          // padding: zero mass, no contribution
        if (p < p1) {
          const float4 v = __ldg(&pos_mass[p]);
          sv = make_float4(v.x - ref.x, v.y - ref.y, v.z - ref.z, v.w);
        }
        ws.src[j * 32 + lane] = sv;
      }
      __syncwarp();
      const int cnt = (int)min((long long)kSrcTile, (p1 - tile + 3) & ~3ll);
#pragma unroll 4
      for (int j = 0; j < cnt; ++j) {
        const float4 sv = ws.src[j];
        const float2 sx = make_float2(sv.x, sv.x), sy = make_float2(sv.y, sv.y), sz = make_float2(sv.z, sv.z);
        const float2 sm = make_float2(sv.w, sv.w);
#pragma unroll
        for (int t = 0; t < 2; ++t) {
          const float2 dx = __fadd2_rn(sx, ntx[t]);
          const float2 dy = __fadd2_rn(sy, nty[t]);
          const float2 dz = __fadd2_rn(sz, ntz[t]);
          float2 u = __ffma2_rn(dx, dx, e2);
          u = __ffma2_rn(dy, dy, u);
          u = __ffma2_rn(dz, dz, u);
          const float2 r = make_float2(mbp_rsqrt(u.x), mbp_rsqrt(u.y));
          phi[t] = __ffma2_rn(r, sm, phi[t]);
        }
      }
    }
#pragma unroll
    for (int t = 0; t < 2; ++t) {
      const long long k0 = tb + t * 64 + lane, k1 = k0 + 32;
      if (k0 < te) asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&phi64[k0]), "d"((double)phi[t].x) : "memory");
      if (k1 < te) asm volatile("red.global.add.f64 [%0], %1;" ::"l"(&phi64[k1]), "d"((double)phi[t].y) : "memory");
    }
  }
}

// phi_i = -(sum - self term); (phi, index) minimum per halo, lowest index on ties.  One CTA per halo (grid-stride).
__global__ void __launch_bounds__(256) k_mbp_reduce(const float4* __restrict__ pos_mass,
                                                     const long long* __restrict__ halo_start, int nhalo, float eps2,
                                                     const double* __restrict__ phi64, float* __restrict__ phi_out,
                                                     long long* __restrict__ mbp_index, float* __restrict__ mbp_phi) {
  __shared__ double s_phi[8];
  __shared__ long long s_idx[8];
  const float rself = mbp_rsqrt(eps2);          // the value the pair loop used for d = 0
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (int h = blockIdx.x; h < nhalo; h += gridDim.x) {
    const long long hb = __ldg(&halo_start[h]), he = __ldg(&halo_start[h + 1]);
    double best = 1.0e300;
    long long bi = -1;
    for (long long i = hb + threadIdx.x; i < he; i += blockDim.x) {
      const float m = __ldg(&pos_mass[i].w);
      const double p = -(phi64[i] - (double)(m * rself));
      if (phi_out) phi_out[i] = (float)p;
      if (p < best) { best = p; bi = i; }         // ascending i per thread: the first minimum is kept
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) {
      const double ob = __shfl_xor_sync(0xffffffffu, best, o);
      const long long oi = __shfl_xor_sync(0xffffffffu, bi, o);
      if (oi >= 0 && (bi < 0 || ob < best || (ob == best && oi < bi))) { best = ob; bi = oi; }
    }
    __syncthreads();
    if (lane == 0) { s_phi[w] = best; s_idx[w] = bi; }
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int k = 1; k < 8; ++k)
        if (s_idx[k] >= 0 && (bi < 0 || s_phi[k] < best || (s_phi[k] == best && s_idx[k] < bi))) { best = s_phi[k]; bi = s_idx[k]; }
      mbp_index[h] = bi;
      if (mbp_phi) mbp_phi[h] = bi >= 0 ? (float)best : 0.f;
    }
  }
}

// items per halo (target tiles x source chunks), before the exclusive scan
__global__ void __launch_bounds__(256) k_mbp_items(const long long* __restrict__ halo_start, int nhalo,
                                                    unsigned long long* __restrict__ items) {
  const int h = blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= nhalo) return;
  const unsigned long long nh = (unsigned long long)(__ldg(&halo_start[h + 1]) - __ldg(&halo_start[h]));
  items[h] = ((nh + kMbpTargets - 1) / kMbpTargets) * ((nh + kMbpChunk - 1) / kMbpChunk);
}

size_t mbp_workspace_layout(int64_t n, int64_t nhalo, size_t* o_phi, size_t* o_prefix, size_t* o_start, size_t* o_tmp) {
  auto up = [](size_t x) { return (x + 255) / 256 * 256; };
  size_t off = 256;                                   // counter block
  *o_phi = off; off = up(off + 8 * (size_t)(n > 0 ? n : 1));
  *o_prefix = off; off = up(off + 8 * (size_t)(nhalo + 1));
  *o_start = off; off = up(off + 8 * (size_t)(nhalo + 1));
  *o_tmp = off; off = up(off + 8 * ((size_t)nhalo / 4096 + 2));
  return off;
}

// The halo table is read from host memory during the call (one pageable->device copy: the runtime stages it before
// returning, so the caller's buffer is free on return); the item prefix is computed on the device.  No stream sync.
cudaError_t launch_mbp(srpp_ctx* c, const float4* pos_mass, int64_t n, const int64_t* halo_start_host, int64_t nhalo,
                       float* phi_out, long long* mbp_index, float* mbp_phi, char* ws) {
  cudaStream_t st = c->stream;
  size_t o_phi, o_prefix, o_start, o_tmp;
  mbp_workspace_layout(n, nhalo, &o_phi, &o_prefix, &o_start, &o_tmp);
  unsigned long long* counter = (unsigned long long*)ws;
  double* phi64 = (double*)(ws + o_phi);
  unsigned long long* prefix = (unsigned long long*)(ws + o_prefix);
  long long* hs = (long long*)(ws + o_start);
  unsigned long long* tmp = (unsigned long long*)(ws + o_tmp);
  cudaError_t e;
  if ((e = cudaMemsetAsync(counter, 0, 256, st)) != cudaSuccess) return e;
  if ((e = cudaMemsetAsync(phi64, 0, 8 * (size_t)(n > 0 ? n : 1), st)) != cudaSuccess) return e;
  if ((e = cudaMemcpyAsync(hs, halo_start_host, 8 * ((size_t)nhalo + 1), cudaMemcpyHostToDevice, st)) != cudaSuccess) return e;
  if (nhalo == 0) return cudaSuccess;
  k_mbp_items<<<(int)((nhalo + 255) / 256), 256, 0, st>>>(hs, (int)nhalo, prefix);
  if ((e = launch_scan_u64(st, prefix, (int)nhalo, tmp, &prefix[nhalo], counter + 8)) != cudaSuccess) return e;
  const float eps2 = c->fc.eps2;
  if (!c->mbp_occ) {
    int occ = 1;
    if ((e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_mbp_phi, kForceThreads, 0)) != cudaSuccess) return e;
    c->mbp_occ = std::max(occ, 1);
  }
  k_mbp_phi<<<c->num_sms * c->mbp_occ, kForceThreads, 0, st>>>(pos_mass, hs, prefix, (int)nhalo, eps2, counter, phi64);
  const int grid = (int)std::min<int64_t>(nhalo, (int64_t)c->num_sms * 8);
  k_mbp_reduce<<<grid, 256, 0, st>>>(pos_mass, hs, (int)nhalo, eps2, phi64, phi_out, mbp_index, mbp_phi);
  c->launches += 6;
  return cudaGetLastError();
}

}  // namespace srpp
