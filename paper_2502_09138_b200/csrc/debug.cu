// debug.cu -- test-only exports of intermediate results (tpc_debug_* in include/tpc_track.h).
// Not on the hot path: these kernels only re-shape what a1..a5 left in the handle's scratch so that the
// parity tests can compare link tables, seeds and tracklets with the oracle element by element.
#include "tpc_internal.cuh"

namespace {

// Links live in sorted space (positions in srt); the exports translate them to cluster ids.
// which = 0: the raw a2 tables.  which = 1: the cleaned links exactly as a3 left them for a4 -- the cleaned up links
// are a3's clean_up table; a3 keeps no down-link table (nothing downstream reads one), so the cleaned
// down links are the inverse of what it wrote (mutuality, P11): dn'[up'[h]] = h.
__global__ void dbg_links_kernel(int64_t n, int which, const int4* __restrict__ srt, const int32_t* __restrict__ up,
                                 const int32_t* __restrict__ dn, const int32_t* __restrict__ clean_up,
                                 int32_t* __restrict__ up_o,
                                 int32_t* __restrict__ dn_o) {
  const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (p >= n) return;
  const int4 c = srt[p];
  if (which == 0) {
    const int u = up[p], d = dn[p];
    up_o[c.z] = u >= 0 ? srt[u].z : -1;
    dn_o[c.z] = d >= 0 ? srt[d].z : -1;
  } else {
    const int cu = clean_up[p];
    up_o[c.z] = cu >= 0 ? srt[cu].z : -1;
    if (cu >= 0) dn_o[srt[cu].z] = c.z;
  }
}

__global__ void dbg_seed_len_kernel(const DevCtl* ctl, const int32_t* __restrict__ seed_start,
                                    const int32_t* __restrict__ seed_pos, const int32_t* __restrict__ clean_up,
                                    int32_t* __restrict__ start, int32_t* __restrict__ len) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= (int64_t)ctl->n_seeds) return;
  int l = 1;
  for (int c = clean_up[seed_pos[i]]; c >= 0; c = clean_up[c]) ++l;
  start[i] = seed_start[i];
  len[i] = l;
}

__global__ void dbg_tracklets_kernel(const DevCtl* ctl, int n_rows, const float4* __restrict__ tl_rec,
                                     const int32_t* __restrict__ tl_hits, const uint32_t* __restrict__ tl_span,
                                     float* par, float* cov, float* chi2,
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
    for (int r = 0; r < n_rows; ++r) {   // only the rows of the visited span hold entries
      const int smin = tl_span[i] & 0xff, smax = (tl_span[i] >> 8) & 0xff;
      hits[i * n_rows + r] = (r >= smin && r <= smax) ? tl_hits[i * n_rows + r] : -1;
    }
}

__global__ void dbg_owner_kernel(int64_t n, const uint32_t* __restrict__ owner, int32_t* __restrict__ out) {
  const int64_t h = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (h >= n) return;
  const uint32_t w = owner[h];
  out[h] = w ? (int32_t)(0xFFFFFFu - (w & 0xFFFFFFu)) : -1;
}

}  // namespace

cudaError_t launch_dbg_links(const tpc_tracker* t, int64_t n, int which, int32_t* up, int32_t* dn, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  if (which == 1) {   // down links are scattered through the inverse: start from "none"
    cudaError_t e = cudaMemsetAsync(dn, 0xff, (size_t)n * 4, st);
    if (e != cudaSuccess) return e;
  }
  dbg_links_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, which, t->s.srt, t->s.link_up, t->s.link_dn, t->s.clean_up, up, dn);
  return cudaGetLastError();
}
cudaError_t launch_dbg_seed_len(const tpc_tracker* t, int32_t* start, int32_t* len, cudaStream_t st) {
  if (t->s_cap == 0) return cudaSuccess;
  dbg_seed_len_kernel<<<(unsigned)((t->s_cap + 255) / 256), 256, 0, st>>>(t->s.ctl, t->s.seed_start, t->s.seed_pos, t->s.clean_up, start, len);
  return cudaGetLastError();
}
cudaError_t launch_dbg_tracklets(const tpc_tracker* t, float* par, float* cov, float* chi2, int32_t* n_hits,
                                 int32_t* hits, cudaStream_t st) {
  if (t->s_cap == 0) return cudaSuccess;
  dbg_tracklets_kernel<<<(unsigned)((t->s_cap + 127) / 128), 128, 0, st>>>(
      t->s.ctl, t->g.n_rows, t->s.tl_rec, t->s.tl_hits, t->s.tl_span, par, cov, chi2, n_hits, hits);
  return cudaGetLastError();
}
cudaError_t launch_dbg_owner(const tpc_tracker* t, int64_t n, int32_t* owner, cudaStream_t st) {
  if (n == 0) return cudaSuccess;
  dbg_owner_kernel<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, t->s.owner, owner);
  return cudaGetLastError();
}
