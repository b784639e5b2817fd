// a8_compress.cu -- NEXT-3: track-model cluster compression, the residual transform (readings P50..P52,
// DESIGN.md; PAPER.md:19 "several processing steps to reduce the TPC data", :29).  tpc_compress / tpc_decompress.
//
// Every cluster an output track owns is replaced by its residual against an integer predictor built from the track's
// previous hits (first difference, two-point line with the row gaps, or the least-squares line through the last four
// hits in consecutive rows), plus the row step.  Integer only -> bit-exact with the oracle, and lossless:
// tpc_decompress rebuilds rows and coordinates.  The entropy coder that would follow is the paper's separate "TPC rANS
// encoding" line (0.10 %); here the residual histograms are produced so that its ideal output size can be stated.
//
// Encoding is parallel over hits: a warp takes a track, lane l the hits j = l, l + 32, ...; a hit's predecessors come
// from the neighbouring lanes by shuffle (and from the previous 32-hit chunk through four carried values).
#include "tpc_internal.cuh"

namespace {

constexpr int A8_THREADS = 256;
constexpr int A8_CENTRAL = 2048;   // residuals in [-1024, 1023] are counted in shared memory first

__device__ __forceinline__ long long floor_div(long long a, long long b) {   // b > 0
  long long q = a / b;
  if ((a % b != 0) && (a < 0)) --q;
  return q;
}

// P50 predictor: c1 = c_{j-1}, c2 = c_{j-2}, c4 = c_{j-4}; four = the last five rows are consecutive
__device__ __forceinline__ int predict(bool four, int c1, int c2, int c4, int g1, int g2) {
  if (four) return (int)floor_div(2ll * c1 + c2 - c4, 2);
  return (int)((long long)c1 + floor_div(((long long)c1 - c2) * g2, g1));
}

__device__ __forceinline__ int pick4(const int a[4], int i) {
  return i == 0 ? a[0] : i == 1 ? a[1] : i == 2 ? a[2] : a[3];
}

__device__ __forceinline__ void count(uint32_t* s_hist, uint32_t* g_hist, int res) {
  const int c = res + A8_CENTRAL / 2;
  if (c >= 0 && c < A8_CENTRAL) atomicAdd(&s_hist[c], 1u);
  else atomicAdd(&g_hist[min(max(res + 32768, 0), 65535)], 1u);   // P52: edge bins collect everything beyond
}

__global__ void __launch_bounds__(A8_THREADS)
a8_compress_kernel(const int32_t* __restrict__ y, const int32_t* __restrict__ z, const uint8_t* __restrict__ hit_row,
                   const tpc_track_rec_t* __restrict__ tracks, int32_t track_capacity,
                   const int32_t* __restrict__ hit_ids, int32_t hit_capacity, const int32_t* __restrict__ counts,
                   uint8_t* __restrict__ drow, int32_t* __restrict__ ry, int32_t* __restrict__ rz,
                   uint32_t* __restrict__ hist_ry, uint32_t* __restrict__ hist_rz, uint32_t* __restrict__ hist_drow) {
  __shared__ uint32_t s_hy[A8_CENTRAL], s_hz[A8_CENTRAL], s_hd[256];
  for (int i = threadIdx.x; i < A8_CENTRAL; i += blockDim.x) s_hy[i] = s_hz[i] = 0;
  for (int i = threadIdx.x; i < 256; i += blockDim.x) s_hd[i] = 0;
  __syncthreads();
  const unsigned FULL = 0xffffffffu;
  const int lane = threadIdx.x & 31;
  const int n_tracks = (counts[1] <= hit_capacity) ? min(counts[0], track_capacity) : 0;
  const int warps = gridDim.x * (blockDim.x >> 5);
  for (int t = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); t < n_tracks; t += warps) {
    const int off = tracks[t].hit_offset, m = tracks[t].n_hits;
    // values carried from the previous chunk of 32 hits: rows and coordinates of hits base-1 .. base-4
    int cr[4] = {0, 0, 0, 0}, cy[4] = {0, 0, 0, 0}, cz[4] = {0, 0, 0, 0};
    for (int base = 0; base < m; base += 32) {
      const int j = base + lane;
      const bool in = j < m;
      int r = 0, vy = 0, vz = 0;
      if (in) {
        const int h = hit_ids[off + j];
        r = hit_row[off + j];
        vy = y[h];
        vz = z[h];
      }
      int pr[4], py[4], pz[4];   // predecessors j-1 .. j-4
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const int sr = __shfl_up_sync(FULL, r, k + 1), sy = __shfl_up_sync(FULL, vy, k + 1), sz = __shfl_up_sync(FULL, vz, k + 1);
        const bool own = lane > k;   // the predecessor is in this chunk; otherwise one of the carried values
        const int ci = k - lane;     // 0..3 when !own (selects, not indexing: the arrays stay in registers)
        pr[k] = own ? sr : pick4(cr, ci);
        py[k] = own ? sy : pick4(cy, ci);
        pz[k] = own ? sz : pick4(cz, ci);
      }
      if (in) {
        int d, resy, resz;
        if (j == 0) {
          d = r; resy = vy; resz = vz;
        } else if (j == 1) {
          d = r - pr[0]; resy = vy - py[0]; resz = vz - pz[0];
        } else {
          const int g2 = r - pr[0], g1 = pr[0] - pr[1];
          const bool four = j >= 4 && g2 == 1 && g1 == 1 && pr[1] - pr[2] == 1 && pr[2] - pr[3] == 1;
          d = g2;
          resy = vy - predict(four, py[0], py[1], py[3], g1, g2);
          resz = vz - predict(four, pz[0], pz[1], pz[3], g1, g2);
          count(s_hy, hist_ry, resy);
          count(s_hz, hist_rz, resz);
        }
        drow[off + j] = (uint8_t)d;
        ry[off + j] = resy;
        rz[off + j] = resz;
        if (j >= 1) atomicAdd(&s_hd[d & 255], 1u);
      }
      // carry the last four hits of this chunk (lanes 31, 30, 29, 28) to the next one
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        cr[k] = __shfl_sync(FULL, r, 31 - k);
        cy[k] = __shfl_sync(FULL, vy, 31 - k);
        cz[k] = __shfl_sync(FULL, vz, 31 - k);
      }
    }
  }
  __syncthreads();
  for (int i = threadIdx.x; i < A8_CENTRAL; i += blockDim.x) {
    if (s_hy[i]) atomicAdd(&hist_ry[i - A8_CENTRAL / 2 + 32768], s_hy[i]);
    if (s_hz[i]) atomicAdd(&hist_rz[i - A8_CENTRAL / 2 + 32768], s_hz[i]);
  }
  for (int i = threadIdx.x; i < 256; i += blockDim.x)
    if (s_hd[i]) atomicAdd(&hist_drow[i], s_hd[i]);
}

// P51: the inverse, one thread per track (each hit needs the rebuilt coordinates of its predecessors).
__global__ void __launch_bounds__(128)
a8_decompress_kernel(const tpc_track_rec_t* __restrict__ tracks, int32_t track_capacity, int32_t hit_capacity,
                     const int32_t* __restrict__ counts, const uint8_t* __restrict__ drow,
                     const int32_t* __restrict__ ry, const int32_t* __restrict__ rz, int32_t* __restrict__ row,
                     int32_t* __restrict__ y, int32_t* __restrict__ z) {
  const int n_tracks = (counts[1] <= hit_capacity) ? min(counts[0], track_capacity) : 0;
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= n_tracks) return;
  const int off = tracks[t].hit_offset, m = tracks[t].n_hits;
  int r1 = 0, r2 = 0, r3 = 0, r4 = 0, y1 = 0, y2 = 0, y3 = 0, y4 = 0, z1 = 0, z2 = 0, z3 = 0, z4 = 0;
  for (int j = 0; j < m; ++j) {
    const int d = drow[off + j], ey = ry[off + j], ez = rz[off + j];
    int r, vy, vz;
    if (j == 0) {
      r = d; vy = ey; vz = ez;
    } else if (j == 1) {
      r = r1 + d; vy = y1 + ey; vz = z1 + ez;
    } else {
      r = r1 + d;
      const int g1 = r1 - r2;
      const bool four = j >= 4 && d == 1 && g1 == 1 && r2 - r3 == 1 && r3 - r4 == 1;
      vy = predict(four, y1, y2, y4, g1, d) + ey;
      vz = predict(four, z1, z2, z4, g1, d) + ez;
    }
    row[off + j] = r;
    y[off + j] = vy;
    z[off + j] = vz;
    r4 = r3; r3 = r2; r2 = r1; r1 = r;
    y4 = y3; y3 = y2; y2 = y1; y1 = vy;
    z4 = z3; z3 = z2; z2 = z1; z1 = vz;
  }
}

}  // namespace

cudaError_t launch_a8_compress(const tpc_tracker* t, const int32_t* y, const int32_t* z, const tpc_tracks_out_t* tracks,
                               const tpc_compressed_t* c, cudaStream_t st) {
  cudaError_t e = cudaMemsetAsync(c->hist_ry, 0, 65536 * 4, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->hist_rz, 0, 65536 * 4, st);
  if (e == cudaSuccess) e = cudaMemsetAsync(c->hist_drow, 0, 256 * 4, st);
  if (e != cudaSuccess || t->last_n == 0 || tracks->track_capacity == 0) return e;
  a8_compress_kernel<<<t->a4_sms * 4, A8_THREADS, 0, st>>>(y, z, t->s.hit_row, tracks->tracks, tracks->track_capacity,
                                                          tracks->hit_ids, tracks->hit_capacity, tracks->counts, c->drow,
                                                          c->ry, c->rz, c->hist_ry, c->hist_rz, c->hist_drow);
  return cudaGetLastError();
}

cudaError_t launch_a8_decompress(const tpc_tracker* t, const tpc_tracks_out_t* tracks, const tpc_compressed_t* c,
                                 int32_t* row, int32_t* y, int32_t* z, cudaStream_t st) {
  (void)t;
  if (tracks->track_capacity == 0) return cudaSuccess;
  a8_decompress_kernel<<<(unsigned)((tracks->track_capacity + 127) / 128), 128, 0, st>>>(
      tracks->tracks, tracks->track_capacity, tracks->hit_capacity, tracks->counts, c->drow, c->ry, c->rz, row, y, z);
  return cudaGetLastError();
}
