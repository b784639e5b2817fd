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
constexpr int A0_PER_THREAD = 8;

// Input contract check (tpc_track.h): row_offsets must be an ascending CSR over exactly n clusters, starting at 0.
// A violation raises ctl->bad_offsets; a0..a3 then return at once (malformed offsets would become out-of-range
// scatter addresses in a1), no seed exists, and a5 reports TPC_FLAG_BAD_OFFSETS with zero tracks.
__global__ void __launch_bounds__(256)
a0_check_kernel(int64_t R, int64_t n, const uint32_t* __restrict__ ro, DevCtl* __restrict__ ctl) {
  bool bad = false;
  for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < R; i += (int64_t)gridDim.x * blockDim.x)
    bad |= ro[i] > ro[i + 1];
  if (blockIdx.x == 0 && threadIdx.x == 0) bad |= ro[0] != 0u || (int64_t)ro[R] != n;
  if (bad) ctl->bad_offsets = 1u;
}

// grid = (chunks, n_sectors): block (c, s) reduces its slice of sector s's contiguous cluster range.
__global__ void __launch_bounds__(A0_THREADS)
a0_origin_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, const int32_t* __restrict__ z,
                 const uint32_t* __restrict__ ro, uint32_t* __restrict__ sec_key) {
  __shared__ int red[A0_THREADS / 32];
  if (ctl->bad_offsets) return;
  for (int sec = blockIdx.y; sec < g.n_sectors; sec += gridDim.y) {   // block-uniform loop (gridDim.y caps at 65535)
  const uint32_t a = ro[(size_t)sec * g.n_rows], b = ro[(size_t)(sec + 1) * g.n_rows];
  int zmin = INT32_MAX;
  for (uint32_t base = a + blockIdx.x * (A0_THREADS * A0_PER_THREAD); base < b;
       base += gridDim.x * (A0_THREADS * A0_PER_THREAD)) {
    int v[A0_PER_THREAD];
#pragma unroll
    for (int k = 0; k < A0_PER_THREAD; ++k) {
      const uint32_t i = base + k * A0_THREADS + threadIdx.x;
      v[k] = i < b ? z[i] : INT32_MAX;
    }
#pragma unroll
    for (int k = 0; k < A0_PER_THREAD; ++k) zmin = min(zmin, v[k]);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) zmin = min(zmin, __shfl_xor_sync(0xffffffffu, zmin, o));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = zmin;
  __syncthreads();
  if (threadIdx.x == 0) {
#pragma unroll
    for (int w = 0; w < A0_THREADS / 32; ++w) zmin = min(zmin, red[w]);
    if (zmin != INT32_MAX) atomicMax(&sec_key[sec], zmin_key(zmin));
  }
  __syncthreads();   // red[] is reused by the next sector
  }
}

// G threads per (sector,row): 32 (a warp per row, 4 rows per block, warp-level sync only) for sparse rows, the whole
// block for long rows.  Bins far outnumber clusters in sparse events, so the per-bin work (zero, scan, write) is
// what a row costs; a warp does it with shuffles and no block barrier.
template <int G>
__device__ __forceinline__ void group_sync() {
  if (G == 32) __syncwarp(); else __syncthreads();
}

template <int G>
__global__ void __launch_bounds__(A1_THREADS)
a1_grid_kernel(const DevGeom g, const DevCtl* __restrict__ ctl, int64_t R, const int32_t* __restrict__ y,
               const int32_t* __restrict__ z, const uint32_t* __restrict__ ro, const uint32_t* __restrict__ sec_key,
               int4* __restrict__ srt, uint32_t* __restrict__ bin_start) {
  extern __shared__ uint32_t hist_all[];
  __shared__ uint32_t wsum[33];
  if (ctl->bad_offsets) return;
  const int grp = threadIdx.x / G, gt = threadIdx.x % G;
  const int64_t sr = (int64_t)blockIdx.x * (A1_THREADS / G) + grp;
  if (sr >= R) return;   // G == 32 only (whole warps); with G == A1_THREADS the grid is exactly R
  uint32_t* const hist = hist_all + (size_t)grp * g.nb_stride;
  const uint32_t a = ro[sr], b = ro[sr + 1];
  const int ny = g.ny, nz = g.nz;
  const int nb = ny * nz;
  const int ymin = g.org_y, zmin = zmin_from_key(sec_key[sr / g.n_rows]);
  for (int k = gt; k < nb; k += G) hist[k] = 0;
  group_sync<G>();

  // pass 1: histogram (the bin index of up to 4 clusters per thread is kept for pass 2)
  constexpr int KEEP = 4;
  int bin[KEEP];
#pragma unroll
  for (int k = 0; k < KEEP; ++k) {
    const uint32_t i = a + k * G + gt;
    bin[k] = -1;
    if (i < b) {
      const int iy = clampi((y[i] - ymin) >> g.shift_y, 0, ny - 1);
      const int iz = clampi((z[i] - zmin) >> g.shift_z, 0, nz - 1);
      bin[k] = iz * ny + iy;
      atomicAdd(&hist[bin[k]], 1u);
    }
  }
  for (uint32_t i = a + KEEP * G + gt; i < b; i += G) {
    const int iy = clampi((y[i] - ymin) >> g.shift_y, 0, ny - 1);
    const int iz = clampi((z[i] - zmin) >> g.shift_z, 0, nz - 1);
    atomicAdd(&hist[iz * ny + iy], 1u);
  }
  group_sync<G>();

  // exclusive scan over bins: each thread owns a contiguous chunk
  const int chunk = (nb + G - 1) / G;
  const int k0 = min(gt * chunk, nb), k1 = min(k0 + chunk, nb);
  uint32_t sum = 0;
  for (int k = k0; k < k1; ++k) sum += hist[k];
  uint32_t run;
  if (G == 32) {
    uint32_t inc = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t t = __shfl_up_sync(0xffffffffu, inc, o);
      if (gt >= o) inc += t;
    }
    run = inc - sum;
  } else {
    uint32_t total;
    run = block_excl_scan(sum, wsum, &total);
  }
  for (int k = k0; k < k1; ++k) {
    const uint32_t c = hist[k];
    hist[k] = run;
    run += c;
  }
  group_sync<G>();
  uint32_t* bs = bin_start + (size_t)sr * g.nb_stride;
  for (int k = gt; k < nb; k += G) bs[k] = a + hist[k];   // coalesced
  if (gt == 0) bs[nb] = b;
  group_sync<G>();

  // pass 2: scatter into bin order (order inside a bin is arbitrary; every consumer breaks ties by id)
#pragma unroll
  for (int k = 0; k < KEEP; ++k) {
    const uint32_t i = a + k * G + gt;
    if (bin[k] >= 0) srt[a + atomicAdd(&hist[bin[k]], 1u)] = make_int4(y[i], z[i], (int32_t)i, 0);
  }
  for (uint32_t i = a + KEEP * G + gt; i < b; i += G) {
    const int yi = y[i], zi = z[i];
    const int iy = clampi((yi - ymin) >> g.shift_y, 0, ny - 1);
    const int iz = clampi((zi - zmin) >> g.shift_z, 0, nz - 1);
    srt[a + atomicAdd(&hist[iz * ny + iy], 1u)] = make_int4(yi, zi, (int32_t)i, 0);
  }
}

}  // namespace

// rows per block and shared memory of the variant chosen for this call
static bool a1_warp_rows(const tpc_tracker* t, int64_t n) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  return t->g.nb_stride <= 4096 && n <= R * 256;   // sparse rows: a warp per row
}

size_t a1_smem_bytes(const DevGeom& g) { return (size_t)(g.nb_stride) * sizeof(uint32_t); }

cudaError_t setup_a1_attributes(const tpc_tracker* t) {
  // the grid shape may change from call to call (api.cu: choose_grid): allow the largest histogram up front
  (void)t;
  cudaError_t e = cudaFuncSetAttribute(a1_grid_kernel<A1_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                       (GRID_MAX_BINS + 4) * (int)sizeof(uint32_t));
  if (e != cudaSuccess) return e;
  return cudaFuncSetAttribute(a1_grid_kernel<32>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                              4096 * (int)sizeof(uint32_t) * (A1_THREADS / 32));
}

cudaError_t launch_a1_grid(const tpc_tracker* t, const int32_t* y, const int32_t* z, const uint32_t* ro, int64_t n,
                           cudaStream_t st) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (R == 0) return cudaSuccess;
  if (a1_warp_rows(t, n)) {
    const int per = A1_THREADS / 32;
    a1_grid_kernel<32><<<(unsigned)((R + per - 1) / per), A1_THREADS, a1_smem_bytes(t->g) * per, st>>>(
        t->g, t->s.ctl, R, y, z, ro, t->s.sec_key, t->s.srt, t->s.bin_start);
  } else {
    a1_grid_kernel<A1_THREADS><<<(unsigned)R, A1_THREADS, a1_smem_bytes(t->g), st>>>(
        t->g, t->s.ctl, R, y, z, ro, t->s.sec_key, t->s.srt, t->s.bin_start);
  }
  return cudaGetLastError();
}

cudaError_t launch_a0_check(const tpc_tracker* t, const uint32_t* ro, int64_t n, cudaStream_t st) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  int64_t blocks = (R + 255) / 256;
  blocks = blocks < 1 ? 1 : (blocks > 1024 ? 1024 : blocks);
  a0_check_kernel<<<(unsigned)blocks, 256, 0, st>>>(R, n, ro, t->s.ctl);
  return cudaGetLastError();
}

cudaError_t launch_a0_origin(const tpc_tracker* t, const int32_t* z, const uint32_t* ro, int64_t n, cudaStream_t st) {
  if (t->g.n_sectors == 0 || n == 0) return cudaSuccess;
  // chunks per sector from the average sector size (a sector larger than that just loops)
  const int64_t per_block = A0_THREADS * A0_PER_THREAD;
  int64_t chunks = (n / t->g.n_sectors + per_block - 1) / per_block;
  if (chunks < 1) chunks = 1;
  if (chunks > 1024) chunks = 1024;
  a0_origin_kernel<<<dim3((unsigned)chunks, (unsigned)(t->g.n_sectors < 65535 ? t->g.n_sectors : 65535)), A0_THREADS, 0, st>>>(t->g, t->s.ctl, z, ro, t->s.sec_key);
  return cudaGetLastError();
}
