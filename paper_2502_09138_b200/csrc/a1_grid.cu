// a1_grid.cu -- stage a1: per-(sector,row) (y,z) grid build by counting sort (north_star
// "a counting-sort/prefix-scan grid build").  The grid is only an accelerator for a2 and a4: the definition of
// both searches is a scan of the whole adjacent row (SURVEY 8(c) "Stage 1-2", P17), so bin size and origin are
// invisible in the results.
//
// a0: one warp per (sector,row) reduces the row's smallest z and atomicMax-es its key into the sector's word, so
// the z origin of a sector's grid follows the data (drift offsets of pile-up collisions cost no bins).  The y
// origin is the geometry's (minus the widest row's half width).
// a1: one CTA per (sector,row):  pass 1 shared-memory histogram over bins (y fastest);  block exclusive scan;  bin
// starts written as global sorted indices;  pass 2 scatter of (y, z, id) as one 16-byte record into bin order.
// Clusters beyond the geometry's nominal extent land in the edge bins (clamp), which keeps both searches exact
// (clamping is monotone, so bin distances never grow).
#include "tpc_internal.cuh"

namespace {

constexpr int A1_THREADS = 128;

__device__ __forceinline__ int clampi(int v, int lo, int hi) { return v < lo ? lo : (v > hi ? hi : v); }

constexpr int A0_THREADS = 256;

__global__ void __launch_bounds__(A0_THREADS)
a0_origin_kernel(const DevGeom g, int64_t R, const int32_t* __restrict__ z, const uint32_t* __restrict__ ro,
                 uint32_t* __restrict__ sec_key) {
  const int64_t sr = (int64_t)blockIdx.x * (A0_THREADS / 32) + (threadIdx.x >> 5);
  if (sr >= R) return;
  const unsigned lane = threadIdx.x & 31;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  if (a == b) return;
  int zmin = INT32_MAX;
  for (uint32_t i = a + lane; i < b; i += 32) zmin = min(zmin, z[i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) zmin = min(zmin, __shfl_xor_sync(0xffffffffu, zmin, o));
  if (lane == 0) atomicMax(&sec_key[sr / g.n_rows], zmin_key(zmin));
}

__global__ void __launch_bounds__(A1_THREADS)
a1_grid_kernel(const DevGeom g, const int32_t* __restrict__ y, const int32_t* __restrict__ z,
               const uint32_t* __restrict__ ro, const uint32_t* __restrict__ sec_key, int4* __restrict__ srt,
               uint32_t* __restrict__ bin_start) {
  extern __shared__ uint32_t hist[];
  __shared__ uint32_t wsum[33];
  const int sr = blockIdx.x;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  const int ny = g.ny, nz = g.nz;
  const int nb = ny * nz;
  const int tid = threadIdx.x;
  const int ymin = g.org_y, zmin = zmin_from_key(sec_key[sr / g.n_rows]);
  for (int k = tid; k < nb; k += A1_THREADS) hist[k] = 0;
  __syncthreads();

  // pass 1: histogram
  for (uint32_t i = a + tid; i < b; i += A1_THREADS) {
    int iy = clampi((y[i] - ymin) >> g.shift_y, 0, ny - 1);
    int iz = clampi((z[i] - zmin) >> g.shift_z, 0, nz - 1);
    atomicAdd(&hist[iz * ny + iy], 1u);
  }
  __syncthreads();

  // exclusive scan over bins: each thread owns a contiguous chunk
  const int chunk = (nb + A1_THREADS - 1) / A1_THREADS;
  const int k0 = min(tid * chunk, nb), k1 = min(k0 + chunk, nb);
  uint32_t s = 0;
  for (int k = k0; k < k1; ++k) s += hist[k];
  uint32_t total;
  uint32_t run = block_excl_scan(s, wsum, &total);
  uint32_t* bs = bin_start + (size_t)sr * g.nb_stride;
  for (int k = k0; k < k1; ++k) {
    uint32_t c = hist[k];
    hist[k] = run;
    bs[k] = a + run;
    run += c;
  }
  if (tid == 0) bs[nb] = b;
  __syncthreads();

  // pass 2: scatter into bin order (order inside a bin is arbitrary; every consumer breaks ties by id)
  for (uint32_t i = a + tid; i < b; i += A1_THREADS) {
    int yi = y[i], zi = z[i];
    int iy = clampi((yi - ymin) >> g.shift_y, 0, ny - 1);
    int iz = clampi((zi - zmin) >> g.shift_z, 0, nz - 1);
    uint32_t pos = a + atomicAdd(&hist[iz * ny + iy], 1u);
    srt[pos] = make_int4(yi, zi, (int32_t)i, 0);
  }
}

}  // namespace

size_t a1_smem_bytes(const DevGeom& g) { return (size_t)(g.nb_stride) * sizeof(uint32_t); }

cudaError_t setup_a1_attributes(const tpc_tracker* t) {
  return cudaFuncSetAttribute(a1_grid_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)a1_smem_bytes(t->g));
}

cudaError_t launch_a1_grid(const tpc_tracker* t, const int32_t* y, const int32_t* z, const uint32_t* ro, int64_t n,
                           cudaStream_t st) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (R == 0) return cudaSuccess;
  a1_grid_kernel<<<(unsigned)R, A1_THREADS, a1_smem_bytes(t->g), st>>>(t->g, y, z, ro, t->s.sec_key, t->s.srt,
                                                                        t->s.bin_start);
  return cudaGetLastError();
}

cudaError_t launch_a0_origin(const tpc_tracker* t, const int32_t* z, const uint32_t* ro, int64_t n, cudaStream_t st) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (R == 0 || n == 0) return cudaSuccess;
  const int per = A0_THREADS / 32;
  a0_origin_kernel<<<(unsigned)((R + per - 1) / per), A0_THREADS, 0, st>>>(t->g, R, z, ro, t->s.sec_key);
  return cudaGetLastError();
}
