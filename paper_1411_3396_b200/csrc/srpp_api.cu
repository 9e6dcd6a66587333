// srpp_api.cu -- the C ABI declared in include/srpp.h: argument validation, workspace carve-up,
// host-side constants (fp64 re-expansion of the polynomial), and the calls into the kernels.
#include <math.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "srpp_internal.cuh"

namespace srpp {

static inline size_t align_up(size_t x, size_t a = 256) { return (x + a - 1) / a * a; }

// Carve the workspace; with ctx == nullptr only the size is computed.
size_t workspace_layout(const srpp_params& p, int64_t n, srpp_ctx* c) {
  const size_t nn = (size_t)(n > 0 ? n : 1);
  const size_t ncells = (size_t)p.ncell[0] * p.ncell[1] * p.ncell[2];
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes); return o; };
  const size_t o_flags = take(sizeof(DevFlags));
  const size_t o_v0 = take(4 * nn), o_v1 = take(4 * nn), o_v2 = take(4 * nn), o_keys = take(4 * nn);
  const size_t o_ctl = take(sort_ctl_bytes());
  const size_t o_ucur = take(unsort_cursor_bytes(n));
  const size_t o_status = take(8 * (size_t)kSortMaxBins * (nn / kPassTile + 1));   // [tiles][bins] look-back words
  const size_t o_cs = take(4 * (ncells + 1));
  const size_t o_sorted = take(16 * nn);
  const size_t o_prefix = take(8 * (ncells + 1));
  const size_t o_tmp = take(8 * ((ncells + 4095) / 4096 + 1));
  const size_t o_acc = take(8 * 3 * nn);
  // sorted-space state of srpp_subcycle and the incremental re-bin
  const size_t o_sorted1 = take(16 * nn), o_vs0 = take(16 * nn), o_vs1 = take(16 * nn);
  const size_t o_pf = take(4 * (nn / 32 + 2)), o_fw = take(4 * (nn / 32 + 2)), o_mmask = take(4 * (nn / 32 + 2)), o_mwp = take(8 * (nn / 32 + 2));
  const size_t o_tm = take(8 * (nn / 1024 + 2)), o_stmp = take(8 * (nn / 32 / 4096 + nn / 1024 / 4096 + 8));
  const size_t mcap = nn / 4 + 1024;
  const size_t o_ms = take(4 * mcap), o_msr = take(4 * mcap), o_mpos = take(16 * mcap), o_mis = take(4 * mcap), o_mss = take(4 * mcap);
  const size_t o_mflags = take(sizeof(DevFlags)), o_mctl = take(sort_ctl_bytes());
  const size_t o_mstatus = take(8 * (size_t)kSortMaxBins * (mcap / kPassTile + 1));
  const size_t o_msorted = take(16 * mcap), o_mtmp = take(16 * mcap), o_mv0 = take(4 * mcap), o_mv1 = take(4 * mcap);
  const size_t o_mkeys = take(4 * mcap), o_mcs = take(4 * (ncells + 1));
  if (c) {
    char* b = c->ws;
    c->flags = (DevFlags*)(b + o_flags);
    c->vals[0] = (uint32_t*)(b + o_v0); c->vals[1] = (uint32_t*)(b + o_v1);
    c->vals_alt = (uint32_t*)(b + o_v2);
    c->keys_buf[0] = (uint32_t*)(b + o_keys); c->keys_buf[1] = nullptr;
    c->sorted_buf[0] = (float4*)(b + o_sorted); c->sorted_buf[1] = (float4*)(b + o_sorted1);
    c->vel_s[0] = (float4*)(b + o_vs0); c->vel_s[1] = (float4*)(b + o_vs1);
    c->prefix_f = (uint32_t*)(b + o_pf); c->flag_words = (uint32_t*)(b + o_fw); c->mover_mask = (uint32_t*)(b + o_mmask);
    c->mover_wprefix = (unsigned long long*)(b + o_mwp); c->tile_movers = (unsigned long long*)(b + o_tm);
    c->sub_scan_tmp = (unsigned long long*)(b + o_stmp);
    c->mover_slots = (uint32_t*)(b + o_ms); c->mover_slot_by_rank = (uint32_t*)(b + o_msr);
    c->mover_pos = (float4*)(b + o_mpos); c->mover_idx_sorted = (uint32_t*)(b + o_mis); c->mover_slot_sorted = (uint32_t*)(b + o_mss);
    c->m_flags = (DevFlags*)(b + o_mflags); c->m_ctl = (uint32_t*)(b + o_mctl);
    if (c->m_status != (unsigned long long*)(b + o_mstatus)) c->status_n_movers = 0;
    c->m_status = (unsigned long long*)(b + o_mstatus);
    c->m_sorted = (float4*)(b + o_msorted); c->m_tmp = (float4*)(b + o_mtmp);
    c->m_vals[0] = (uint32_t*)(b + o_mv0); c->m_vals[1] = (uint32_t*)(b + o_mv1);
    c->m_keys = (uint32_t*)(b + o_mkeys); c->m_cell_start = (uint32_t*)(b + o_mcs);
    c->m_cap = (int64_t)mcap;
    c->sort_ctl = (uint32_t*)(b + o_ctl);
    c->unsort_cursor = (uint32_t*)(b + o_ucur);
    if (c->sort_status != (unsigned long long*)(b + o_status)) c->status_n = 0;   // the array moved: clear before use
    c->sort_status = (unsigned long long*)(b + o_status);
    c->cell_start = (uint32_t*)(b + o_cs);
    c->sorted = (float4*)(b + o_sorted);
    c->item_prefix = (unsigned long long*)(b + o_prefix);
    c->scan_tmp = (unsigned long long*)(b + o_tmp);
    c->acc64 = (double*)(b + o_acc);
    c->pos_tmp = (float4*)(b + o_acc);
  }
  return off;
}

static int32_t validate(const srpp_params* p) {
  if (!p) return SRPP_ERR_INVALID_ARG;
  for (int a = 0; a < 3; ++a)
    if (!(p->box[a] > 0.f) || !isfinite(p->box[a])) return SRPP_ERR_INVALID_ARG;
  // the force kernel stages coordinates relative to INTEGER reference points (exact periodic shifts in fp32): the box
  // and the cutoff must stay inside fp32's exact-integer range
  for (int a = 0; a < 3; ++a)
    if (p->box[a] > 16777216.f) return SRPP_ERR_GEOMETRY;
  if (!(p->rcut > 0.f) || !isfinite(p->rcut) || !(p->eps > 0.f) || !isfinite(p->eps)) return SRPP_ERR_INVALID_ARG;
  if (p->rcut > 16777216.f) return SRPP_ERR_GEOMETRY;
  for (int k = 0; k < 6; ++k)
    if (!isfinite(p->poly[k])) return SRPP_ERR_INVALID_ARG;
  int64_t ncells = 1;
  for (int a = 0; a < 3; ++a) {
    if (p->ncell[a] < 3) return SRPP_ERR_GEOMETRY;             // 27-cell stencil needs 3 distinct cells (R8)
    if ((double)p->box[a] / (double)p->ncell[a] < (double)p->rcut) return SRPP_ERR_GEOMETRY;
    ncells *= p->ncell[a];
    if (ncells > (1 << 24)) return SRPP_ERR_GEOMETRY;
  }
  return SRPP_OK;
}

// float4 arrays must be 16-byte aligned (vector loads/stores, cp.async 16): a misaligned pointer would raise a sticky
// misaligned-address fault instead of a status code
static inline bool misaligned16(const void* p) { return ((uintptr_t)p & 15u) != 0; }

// Every compute call runs on the device that was current at srpp_create (kernel attributes and occupancy are cached
// per context): a different current device is a state error, not a silent launch on the wrong GPU.
static int32_t check_device(const srpp_ctx* c) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return SRPP_ERR_CUDA;
  return dev == c->device ? SRPP_OK : SRPP_ERR_STATE;
}

static int32_t cuda_fail(srpp_ctx* c, cudaError_t e) {
  if (c) snprintf(c->cuda_err, sizeof(c->cuda_err), "%s: %s", cudaGetErrorName(e), cudaGetErrorString(e));
  return SRPP_ERR_CUDA;
}

}  // namespace srpp

using namespace srpp;

extern "C" {

int32_t srpp_version(void) { return SRPP_VERSION; }

int32_t srpp_default_poly(float* poly_host) {
  if (!poly_host) return SRPP_ERR_INVALID_ARG;
  // SURVEY.md Appendix A (reading R4): fp32 bit patterns of the constrained least-squares fit
  static const uint32_t bits[6] = {0x3EDEAD5Du, 0xBE36288Au, 0x3D2403BCu, 0xBBB0860Au, 0x39CFCFAAu, 0xB74AC976u};
  memcpy(poly_host, bits, sizeof(bits));
  return SRPP_OK;
}

int32_t srpp_workspace_bytes(const srpp_params* params, int64_t n, size_t* bytes_host) {
  if (!bytes_host) return SRPP_ERR_INVALID_ARG;
  const int32_t v = validate(params);
  if (v != SRPP_OK) return v;
  if (n < 0 || n >= ((int64_t)1 << 31)) return SRPP_ERR_INVALID_ARG;
  *bytes_host = workspace_layout(*params, n, nullptr);
  return SRPP_OK;
}

int32_t srpp_create(srpp_ctx** out, const srpp_params* params, void* workspace, size_t workspace_bytes,
                    void* cuda_stream) {
  if (!out) return SRPP_ERR_INVALID_ARG;
  *out = nullptr;
  const int32_t v = validate(params);
  if (v != SRPP_OK) return v;
  if (!workspace) return SRPP_ERR_INVALID_ARG;
  if (((uintptr_t)workspace & 255u) != 0) return SRPP_ERR_WORKSPACE;
  if (workspace_bytes < workspace_layout(*params, 0, nullptr)) return SRPP_ERR_WORKSPACE;
  srpp_ctx* c = new (std::nothrow) srpp_ctx();
  if (!c) return SRPP_ERR_INVALID_ARG;
  memset(c, 0, sizeof(*c));
  c->params = *params;
  c->stream = (cudaStream_t)cuda_stream;
  c->ws = (char*)workspace;
  c->ws_bytes = workspace_bytes;
  c->n = -1;
  cudaError_t e = cudaGetDevice(&c->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->num_sms, cudaDevAttrMultiProcessorCount, c->device);
  if (e != cudaSuccess) { delete c; return SRPP_ERR_CUDA; }
  query_force_occupancy(c->force_blocks_per_sm);

  Geometry& g = c->geo;
  int64_t ncells = 1;
  for (int a = 0; a < 3; ++a) {
    g.box[a] = params->box[a];
    g.ncell[a] = params->ncell[a];
    g.inv_cell[a] = (float)params->ncell[a] / params->box[a];   // one IEEE fp32 division (R10)
    g.cell_w[a] = params->box[a] / (float)params->ncell[a];
    ncells *= params->ncell[a];
    g.periodic[a] = 1;
    g.act_lo[a] = 0;
    g.act_hi[a] = params->ncell[a];
  }
  g.ncells = (int32_t)ncells;
  plan_sort(g.ncells, &c->sort_passes, &c->sort_digit_bits);

  // force constants, in fp64: u = s + eps2 with eps2 the fp32 value the kernel adds, Q(u) = P(u - eps2)
  const double e2 = (double)params->eps * (double)params->eps;
  c->fc.eps2 = (float)e2;
  const double e2f = (double)c->fc.eps2;
  c->fc.rc2e = (float)((double)params->rcut * (double)params->rcut + e2f);
  {  // padding coordinate of empty target / source slots: farther than rc from every real relative coordinate
     // (targets lie within [0, cell_w + 1] of their reference point, sources within [-cell_w - 1, 2 cell_w + 2])
    float wmax = 0.f;
    for (int a = 0; a < 3; ++a) wmax = fmaxf(wmax, params->box[a] / (float)params->ncell[a]);
    c->fc.pad = 8.f * wmax + 4.f * params->rcut + 16.f;
  }
  double q[6];
  for (int k = 0; k < 6; ++k) {
    double acc = 0.0, binom = 1.0, powr = 1.0;   // sum_{j>=k} c_j C(j,k) (-e2f)^(j-k)
    for (int j = k; j < 6; ++j) {
      acc += (double)params->poly[j] * binom * powr;
      binom = binom * (double)(j + 1) / (double)(j + 1 - k);
      powr *= -e2f;
    }
    q[k] = acc;
  }
  // Round -Q's coefficients to fp32.  Plain rounding leaves |Q~ - Q| up to ~4e-7 near the cutoff (the u^k
  // amplify each half-ulp), where f itself is only ~1e-5, so pick, among the 3^6 neighbours within one ulp,
  // the set that minimises max |Q~(u) - Q(u)| over the outer part of the range (where |f| is small).
  float base[6], best[6];
  for (int k = 0; k < 6; ++k) best[k] = base[k] = (float)(-q[k]);
  const double u_hi = (double)c->fc.rc2e, u_lo = u_hi / 3.0;
  double best_err = INFINITY;
  for (int code = 0; code < 729; ++code) {
    float cand[6];
    int t = code;
    for (int k = 0; k < 6; ++k, t /= 3) {
      const int d = t % 3 - 1;
      cand[k] = d == 0 ? base[k] : nextafterf(base[k], d > 0 ? INFINITY : -INFINITY);
    }
    double worst = 0.0;
    for (int i = 0; i <= 64; ++i) {
      const double u = u_lo + (u_hi - u_lo) * i / 64.0;
      double e = 0.0;
      for (int k = 5; k >= 0; --k) e = e * u + ((double)cand[k] + q[k]);
      worst = fmax(worst, fabs(e));
    }
    if (worst < best_err) { best_err = worst; memcpy(best, cand, sizeof(best)); }
  }
  for (int k = 0; k < 6; ++k) c->fc.nq[k] = best[k];
  *out = c;
  return SRPP_OK;
}

void srpp_destroy(srpp_ctx* c) {
  if (!c) return;
  for (int i = 0; i < kNumEvents; ++i)
    if (c->ev[i]) cudaEventDestroy(c->ev[i]);
  for (int i = 0; i < 2; ++i)
    if (c->ev_sub[i]) cudaEventDestroy(c->ev_sub[i]);
  for (int i = 0; i < 3; ++i)
    if (c->ev_copy[i]) cudaEventDestroy(c->ev_copy[i]);
  if (c->copy_stream) cudaStreamDestroy(c->copy_stream);
  free_block_plan(c);
  delete c;
}

int32_t srpp_set_timing(srpp_ctx* c, int32_t enable) {
  if (!c) return SRPP_ERR_INVALID_ARG;
  if (enable) {
    for (int i = 0; i < kNumEvents; ++i)
      if (!c->ev[i]) {
        const cudaError_t e = cudaEventCreate(&c->ev[i]);
        if (e != cudaSuccess) return cuda_fail(c, e);
      }
  }
  c->timing = enable != 0;
  c->ev_mesh_valid = c->ev_accel_valid = false;
  return SRPP_OK;
}

int32_t srpp_get_timings(srpp_ctx* c, srpp_timings* t) {
  if (!c || !t) return SRPP_ERR_INVALID_ARG;
  t->mesh_ms = t->accel_ms = t->force_ms = -1.0f;
  t->rebin_ms = c->rebin_count ? c->rebin_ms_sum / (float)c->rebin_count : -1.0f;
  t->kick_stream_ms = c->rebin_count ? c->subkick_ms_sum / (float)c->rebin_count : -1.0f;
  if (!c->timing) return SRPP_ERR_STATE;
  cudaError_t e = cudaStreamSynchronize(c->stream);
  if (e == cudaSuccess && c->ev_mesh_valid) e = cudaEventElapsedTime(&t->mesh_ms, c->ev[kEvMesh0], c->ev[kEvMesh1]);
  if (e == cudaSuccess && c->ev_accel_valid) {
    e = cudaEventElapsedTime(&t->accel_ms, c->ev[kEvAccel0], c->ev[kEvAccel1]);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&t->force_ms, c->ev[kEvForce0], c->ev[kEvForce1]);
  }
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

int32_t srpp_probe_fp32(srpp_ctx* c, int32_t variant, int32_t trips, double* flops_per_s_host) {
  if (!c || !flops_per_s_host || variant < 0 || variant > 3 || trips < 1) return SRPP_ERR_INVALID_ARG;
  // scratch word: the unused tail of the 256-byte flag block at the head of the workspace
  static_assert(sizeof(DevFlags) <= 128, "flag block layout");
  const cudaError_t e = run_fp32_probe(c->stream, variant, trips, flops_per_s_host, (float*)(c->ws + 128));
  if (e != cudaSuccess) return cuda_fail(c, e);
  c->launches += 2;
  return SRPP_OK;
}

int32_t srpp_set_boundary(srpp_ctx* c, const int32_t* periodic_host, const float* active_lo_host,
                          const float* active_hi_host) {
  if (!c) return SRPP_ERR_INVALID_ARG;
  Geometry& g = c->geo;
  int32_t per[3], clo[3], chi[3];       // validated into temporaries: the boundary is unchanged on error
  for (int a = 0; a < 3; ++a) {
    per[a] = periodic_host ? (periodic_host[a] != 0) : 1;
    float lo = active_lo_host ? active_lo_host[a] : 0.f, hi = active_hi_host ? active_hi_host[a] : c->params.box[a];
    if (!(lo <= hi) || !isfinite(lo) || !isfinite(hi)) return SRPP_ERR_INVALID_ARG;
    lo = fmaxf(lo, 0.f);
    hi = fminf(hi, c->params.box[a]);
    // cells [clo, chi) that can hold a particle with lo <= x < hi: the fp32 cell function of A1 (R10) is monotonic
    // in x, so the cells of lo and of the largest float below hi bound the range
    clo[a] = (int32_t)floorf(lo * g.inv_cell[a]);
    chi[a] = (int32_t)floorf(nextafterf(hi, -INFINITY) * g.inv_cell[a]) + 1;
    if (clo[a] > g.ncell[a] - 1) clo[a] = g.ncell[a] - 1;
    if (clo[a] < 0) clo[a] = 0;
    if (chi[a] > g.ncell[a]) chi[a] = g.ncell[a];
    if (hi <= lo) chi[a] = clo[a];
  }
  for (int a = 0; a < 3; ++a) {
    g.periodic[a] = per[a];
    g.act_lo[a] = clo[a];
    g.act_hi[a] = chi[a];
  }
  return SRPP_OK;
}

int32_t srpp_mbp_workspace_bytes(int64_t n, int64_t nhalo, size_t* bytes_host) {
  if (!bytes_host || n < 0 || n >= ((int64_t)1 << 31) || nhalo < 0 || nhalo > ((int64_t)1 << 24)) return SRPP_ERR_INVALID_ARG;
  size_t a, b, d, t;
  *bytes_host = mbp_workspace_layout(n, nhalo, &a, &b, &d, &t);
  return SRPP_OK;
}

int32_t srpp_mbp(srpp_ctx* c, const float* pos_mass, int64_t n, const int64_t* halo_start_host, int64_t nhalo,
                 float* phi, int64_t* mbp_index, float* mbp_phi, void* workspace, size_t workspace_bytes) {
  if (!c || n < 0 || n >= ((int64_t)1 << 31) || nhalo < 0 || nhalo > ((int64_t)1 << 24) || !halo_start_host ||
      (n > 0 && !pos_mass) || (nhalo > 0 && !mbp_index) || !workspace || misaligned16(pos_mass))
    return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  if (halo_start_host[0] < 0 || halo_start_host[nhalo] > n) return SRPP_ERR_INVALID_ARG;
  for (int64_t h = 0; h < nhalo; ++h)
    if (halo_start_host[h + 1] < halo_start_host[h]) return SRPP_ERR_INVALID_ARG;
  size_t a, b, d, t;
  if (((uintptr_t)workspace & 255u) != 0 || workspace_bytes < mbp_workspace_layout(n, nhalo, &a, &b, &d, &t)) return SRPP_ERR_WORKSPACE;
  const cudaError_t e = launch_mbp(c, (const float4*)pos_mass, n, halo_start_host, nhalo, phi, (long long*)mbp_index,
                                   mbp_phi, (char*)workspace);
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

int32_t srpp_build_mesh(srpp_ctx* c, const float* pos_mass, int64_t n) {
  if (!c || n < 0 || n >= ((int64_t)1 << 31) || (n > 0 && !pos_mass) || misaligned16(pos_mass)) return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  c->n = -1;
  if (workspace_layout(c->params, n, nullptr) > c->ws_bytes) return SRPP_ERR_WORKSPACE;
  workspace_layout(c->params, n, c);
  cudaError_t e = launch_build_mesh(c, (const float4*)pos_mass, n);
  if (e != cudaSuccess) return cuda_fail(c, e);
  float m0 = 1.0f;
  if (n > 0) e = cudaMemcpyAsync(&m0, pos_mass + 3, sizeof(float), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(&c->flags_host, c->flags, sizeof(DevFlags), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return cuda_fail(c, e);
  if (c->flags_host.domain_error) return SRPP_ERR_DOMAIN;
  c->uniform_mass = (c->flags_host.mass_nonuniform == 0);
  c->mass0 = m0;
  c->n = n;
  return SRPP_OK;
}

int32_t srpp_get_mesh(const srpp_ctx* c, const uint32_t** cell_start, const uint32_t** perm, const float** sorted) {
  if (!c) return SRPP_ERR_INVALID_ARG;
  if (c->n < 0) return SRPP_ERR_STATE;
  if (cell_start) *cell_start = c->cell_start;
  if (perm) *perm = c->perm;
  if (sorted) *sorted = (const float*)c->sorted;
  return SRPP_OK;
}

int32_t srpp_accel(srpp_ctx* c, float* acc) {
  if (!c) return SRPP_ERR_INVALID_ARG;
  if (c->n < 0) return SRPP_ERR_STATE;
  if ((c->n > 0 && !acc) || misaligned16(acc)) return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  const cudaError_t e = launch_accel(c, (float4*)acc);
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

int32_t srpp_accel_kick(srpp_ctx* c, float* acc, float* vel, float kdt) {
  if (!c) return SRPP_ERR_INVALID_ARG;
  if (c->n < 0) return SRPP_ERR_STATE;
  if ((c->n > 0 && (!acc || !vel)) || misaligned16(acc) || misaligned16(vel) || !isfinite(kdt)) return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  const cudaError_t e = launch_accel(c, (float4*)acc, (float4*)vel, kdt);
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

int32_t srpp_get_stats(srpp_ctx* c, srpp_stats* s) {
  if (!c || !s) return SRPP_ERR_INVALID_ARG;
  if (c->n < 0) return SRPP_ERR_STATE;
  cudaError_t e = cudaMemcpyAsync(&c->flags_host, c->flags, sizeof(DevFlags), cudaMemcpyDeviceToHost, c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->stream);
  if (e != cudaSuccess) return cuda_fail(c, e);
  s->work_items = c->flags_host.total_items;
  s->pair_slots = c->flags_host.pair_slots;
  s->candidate_pairs = c->flags_host.candidate_pairs;
  s->max_cell_count = c->flags_host.max_cell_count;
  s->uniform_mass = c->uniform_mass ? 1u : 0u;
  s->kernel_launches = c->launches;
  s->rebins_incremental = c->rebin_incremental;
  s->rebins_full = c->rebin_full;
  s->last_movers = c->last_movers;
  return SRPP_OK;
}

int32_t srpp_kick(srpp_ctx* c, float* vel, const float* acc, float kdt, int64_t n) {
  if (!c || n < 0 || (n > 0 && (!vel || !acc)) || !isfinite(kdt) || misaligned16(vel) || misaligned16(acc)) return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  const cudaError_t e = launch_kick(c, (float4*)vel, (const float4*)acc, kdt, n);
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

int32_t srpp_stream(srpp_ctx* c, float* pos_mass, const float* vel, float dt, int64_t n) {
  if (!c || n < 0 || (n > 0 && (!pos_mass || !vel)) || !isfinite(dt) || misaligned16(pos_mass) || misaligned16(vel)) return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  const cudaError_t e = launch_stream(c, (float4*)pos_mass, (const float4*)vel, dt, n);
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

int32_t srpp_step_host(srpp_ctx* c, const float* pos_mass_host, float* vel_host, float* acc_host, float kdt,
                       int64_t n, void* device_scratch, size_t device_scratch_bytes) {
  if (!c || n < 0 || n >= ((int64_t)1 << 31) || (n > 0 && (!pos_mass_host || !acc_host || !device_scratch))) return SRPP_ERR_INVALID_ARG;
  if (const int32_t d = check_device(c)) return d;
  const size_t bytes = 16 * (size_t)n;
  if (device_scratch_bytes < 3 * bytes || ((uintptr_t)device_scratch & 15u)) return SRPP_ERR_WORKSPACE;
  float* d_pos = (float*)device_scratch;
  float* d_acc = (float*)((char*)device_scratch + bytes);
  float* d_vel = (float*)((char*)device_scratch + 2 * bytes);
  // Copies overlap the kernels: the velocities travel on a second stream while the mesh is built and the forces are
  // evaluated (they are needed only by the kick), and the accelerations travel back while the kick runs.
  cudaError_t e = cudaSuccess;
  if (!c->copy_stream) {
    e = cudaStreamCreateWithFlags(&c->copy_stream, cudaStreamNonBlocking);
    for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&c->ev_copy[i], cudaEventDisableTiming);
    if (e != cudaSuccess) return cuda_fail(c, e);
  }
  e = cudaEventRecord(c->ev_copy[0], c->stream);                  // the previous use of the scratch is over
  if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, c->ev_copy[0], 0);
  if (e == cudaSuccess) e = cudaMemcpyAsync(d_pos, pos_mass_host, bytes, cudaMemcpyHostToDevice, c->stream);
  if (e == cudaSuccess && vel_host) {
    e = cudaMemcpyAsync(d_vel, vel_host, bytes, cudaMemcpyHostToDevice, c->copy_stream);
    if (e == cudaSuccess) e = cudaEventRecord(c->ev_copy[1], c->copy_stream);
  }
  if (e != cudaSuccess) return cuda_fail(c, e);
  int32_t rc = srpp_build_mesh(c, d_pos, n);
  if (rc != SRPP_OK) { cudaStreamSynchronize(c->copy_stream); return rc; }
  if (n > 0) {
    // force kernel, then the write-back with the kick fused into it (A6 + A7 in one pass over acc and vel)
    if (c->timing) cudaEventRecord(c->ev[kEvAccel0], c->stream);
    e = launch_accel_sorted(c);
    if (e == cudaSuccess && vel_host) e = cudaStreamWaitEvent(c->stream, c->ev_copy[1], 0);     // velocities have arrived
    if (e == cudaSuccess) e = launch_write_back(c, (float4*)d_acc, vel_host ? (float4*)d_vel : nullptr, kdt);
    if (c->timing) { cudaEventRecord(c->ev[kEvAccel1], c->stream); c->ev_accel_valid = true; }
    if (e != cudaSuccess) { cudaStreamSynchronize(c->copy_stream); return cuda_fail(c, e); }
  }
  // the two downloads run side by side: accelerations on the copy stream, velocities on the solver's stream
  e = cudaEventRecord(c->ev_copy[2], c->stream);
  if (e == cudaSuccess) e = cudaStreamWaitEvent(c->copy_stream, c->ev_copy[2], 0);
  if (e == cudaSuccess) e = cudaMemcpyAsync(acc_host, d_acc, bytes, cudaMemcpyDeviceToHost, c->copy_stream);
  if (e == cudaSuccess && vel_host) e = cudaMemcpyAsync(vel_host, d_vel, bytes, cudaMemcpyDeviceToHost, c->stream);
  if (e != cudaSuccess) return cuda_fail(c, e);
  e = cudaStreamSynchronize(c->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(c->copy_stream);
  return e == cudaSuccess ? SRPP_OK : cuda_fail(c, e);
}

const char* srpp_strerror(int32_t s) {
  switch (s) {
    case SRPP_OK: return "ok";
    case SRPP_ERR_INVALID_ARG: return "invalid argument";
    case SRPP_ERR_GEOMETRY: return "geometry: need ncell >= 3, box/ncell >= rcut, <= 2^24 cells";
    case SRPP_ERR_DOMAIN: return "domain: a position is outside [0, L) or not finite";
    case SRPP_ERR_WORKSPACE: return "workspace too small or misaligned";
    case SRPP_ERR_STATE: return "state: no valid chaining mesh (call srpp_build_mesh first)";
    case SRPP_ERR_CUDA: return "CUDA runtime error";
    case SRPP_ERR_LIMIT: return "limit: size beyond the capacity of the built-in scratch array (srpp_mbp_static)";
    default: return "unknown status";
  }
}

const char* srpp_last_cuda_error(const srpp_ctx* c) { return c ? c->cuda_err : ""; }

}  // extern "C"
