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
#include <math.h>
#include <string.h>

#include <algorithm>
#include <mutex>

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

// --------------------------------------------------------------- srpp_mbp_static: no allocation --
// The same launch sequence as srpp_mbp (launch_mbp above, unchanged), for callers that cannot allocate device memory:
// the workspace is a static __device__ array of this translation unit instead of a caller allocation.  Capacity:
// SRPP_MBP_STATIC_MAX_N members and SRPP_MBP_STATIC_MAX_HALOS halos (include/srpp.h), laid out by mbp_workspace_layout.
constexpr size_t mbp_up256(size_t x) { return (x + 255) / 256 * 256; }
constexpr size_t kMbpStaticBytes = 256 + mbp_up256(8 * (size_t)SRPP_MBP_STATIC_MAX_N) +
                                   2 * mbp_up256(8 * ((size_t)SRPP_MBP_STATIC_MAX_HALOS + 1)) +
                                   mbp_up256(8 * ((size_t)SRPP_MBP_STATIC_MAX_HALOS / 4096 + 2));

// ~9.1 MB on every GPU that loads the library, until the process exits.  In HOST code this name is only a stand-in for
// the symbol, not a device address: the address is looked up once per device with cudaGetSymbolAddress (below).
static __device__ __align__(256) unsigned char g_mbp_static_scratch[kMbpStaticBytes];

namespace {

constexpr int kMbpStaticMaxDevices = 64;
struct MbpStaticDevice {
  char* ws;        // device address of g_mbp_static_scratch on this device
  int num_sms;
  int occ;         // resident CTAs per SM of k_mbp_phi (0 = not queried yet)
  bool ready;
};
MbpStaticDevice g_mbp_static_dev[kMbpStaticMaxDevices];
std::mutex g_mbp_static_mutex;

}  // namespace

extern "C" int32_t srpp_mbp_static(const float* pos_mass, int64_t n, const int64_t* halo_start_host, int64_t nhalo, float eps,
                                   float* phi, int64_t* mbp_index, float* mbp_phi, void* cuda_stream) {
  if (n < 0 || nhalo < 0 || !halo_start_host || (n > 0 && !pos_mass) || (nhalo > 0 && !mbp_index) ||
      ((uintptr_t)pos_mass & 15u) != 0 || !(eps > 0.f) || !isfinite(eps))
    return SRPP_ERR_INVALID_ARG;
  if (n > (int64_t)SRPP_MBP_STATIC_MAX_N || nhalo > (int64_t)SRPP_MBP_STATIC_MAX_HALOS) return SRPP_ERR_LIMIT;
  if (halo_start_host[0] < 0 || halo_start_host[nhalo] > n) return SRPP_ERR_INVALID_ARG;
  for (int64_t h = 0; h < nhalo; ++h)
    if (halo_start_host[h + 1] < halo_start_host[h]) return SRPP_ERR_INVALID_ARG;
  size_t a, b, d, t;
  if (srpp::mbp_workspace_layout(n, nhalo, &a, &b, &d, &t) > kMbpStaticBytes) return SRPP_ERR_LIMIT;   // (cannot happen below the maxima)

  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return SRPP_ERR_CUDA;
  if (dev < 0 || dev >= kMbpStaticMaxDevices) return SRPP_ERR_STATE;
  MbpStaticDevice info;
  {
    // set-up, once per device, with that device current: the array's device address, the SM count
    std::lock_guard<std::mutex> lock(g_mbp_static_mutex);
    MbpStaticDevice& s = g_mbp_static_dev[dev];
    if (!s.ready) {
      char* ptr = nullptr;
      if (cudaGetSymbolAddress((void**)&ptr, g_mbp_static_scratch) != cudaSuccess || !ptr) return SRPP_ERR_CUDA;
      int sms = 0;
      if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1) return SRPP_ERR_CUDA;
      s.ws = ptr;
      s.num_sms = sms;
      s.occ = 0;
      s.ready = true;
    }
    info = s;
  }

  // launch_mbp reads only these fields of a context: stream, eps^2, SM count, cached occupancy, launch counter
  srpp_ctx tmp;
  memset(&tmp, 0, sizeof(tmp));
  tmp.stream = (cudaStream_t)cuda_stream;
  tmp.device = dev;
  tmp.num_sms = info.num_sms;
  tmp.mbp_occ = info.occ;
  tmp.fc.eps2 = (float)((double)eps * (double)eps);      // as srpp_create computes it
  const cudaError_t e = srpp::launch_mbp(&tmp, (const float4*)pos_mass, n, halo_start_host, nhalo, phi, (long long*)mbp_index,
                                         mbp_phi, info.ws);
  if (e != cudaSuccess) return SRPP_ERR_CUDA;
  if (!info.occ && tmp.mbp_occ) {
    std::lock_guard<std::mutex> lock(g_mbp_static_mutex);
    g_mbp_static_dev[dev].occ = tmp.mbp_occ;
  }
  return SRPP_OK;
}
