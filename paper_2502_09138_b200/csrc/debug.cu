// debug.cu -- test-only exports of intermediate results (tpc_debug_* in include/tpc_track.h).
// Not on the hot path: these kernels only re-shape what a1..a5 left in the handle's scratch so that the
// parity tests can compare link tables, seeds and tracklets with the oracle element by element.
#include "tpc_internal.cuh"

namespace {

// Cleaned links exactly as a3 left them for a4: rec[h] = (y, z, cleaned up link, cleaned down link).
__global__ void dbg_clean_kernel(int64_t n, const int4* __restrict__ rec, int32_t* __restrict__ up_o,
                                 int32_t* __restrict__ dn_o) {
  const int64_t h = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n) return;
  const int4 r = rec[h];
  up_o[h] = r.z;
  dn_o[h] = r.w;
}

__global__ void dbg_seed_len_kernel(const DevCtl* ctl, const int32_t* __restrict__ seed_start,
                                    const int4* __restrict__ rec, int32_t* __restrict__ start,
                                    int32_t* __restrict__ len) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)ctl->n_seeds) return;
  const int h0 = seed_start[i];
  int l = 1;
  for (int c = rec[h0].z; c >= 0; c = rec[c].z) ++l;
  start[i] = h0;
  len[i] = l;
}

__global__ void dbg_tracklets_kernel(const DevCtl* ctl, int n_rows, const float4* __restrict__ tl_rec,
                                     const int32_t* __restrict__ tl_hits, float* par, float* cov, float* chi2,
                                     int32_t* n_hits, int32_t* hits) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)ctl->n_seeds) return;
  const float* q = (const float*)(tl_rec + i * TL_REC_V4);
  if (par)
    for (int k = 0; k < 6; ++k) par[i * 6 + k] = q[k];
  if (cov)
    for (int k = 0; k < 15; ++k) cov[i * 15 + k] = q[8 + k];
  if (chi2) chi2[i] = q[6];
  if (n_hits) n_hits[i] = __float_as_int(q[7]);
  if (hits)
    for (int r = 0; r < n_rows; ++r) hits[i * n_rows + r] = tl_hits[i * n_rows + r];
}

__global__ void dbg_owner_kernel(int64_t n, const uint32_t* __restrict__ owner, int32_t* __restrict__ out) {
  const int64_t h = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n) return;
  const uint32_t w = owner[h];
  out[h] = w ? (int32_t)(0xFFFFFFu - (w & 0xFFFFFFu)) : -1;
}

}  // namespace

cudaError_t launch_dbg_clean(const tpc_tracker* t, int64_t n, int32_t* up, int32_t* dn, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  dbg_clean_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, t->s.rec, up, dn);
  return cudaGetLastError();
}
cudaError_t launch_dbg_seed_len(const tpc_tracker* t, int32_t* start, int32_t* len, cudaStream_t st) {
  if (t->s_cap == 0) return cudaSuccess;
  dbg_seed_len_kernel<<<(unsigned)((t->s_cap + 255) / 256), 256, 0, st>>>(t->s.ctl, t->s.seed_start, t->s.rec, start, len);
  return cudaGetLastError();
}
cudaError_t launch_dbg_tracklets(const tpc_tracker* t, float* par, float* cov, float* chi2, int32_t* n_hits,
                                 int32_t* hits, cudaStream_t st) {
  if (t->s_cap == 0) return cudaSuccess;
  dbg_tracklets_kernel<<<(unsigned)((t->s_cap + 127) / 128), 128, 0, st>>>(
      t->s.ctl, t->g.n_rows, t->s.tl_rec, t->s.tl_hits, par, cov, chi2, n_hits, hits);
  return cudaGetLastError();
}
cudaError_t launch_dbg_owner(const tpc_tracker* t, int64_t n, int32_t* owner, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  dbg_owner_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, t->s.owner, owner);
  return cudaGetLastError();
}
