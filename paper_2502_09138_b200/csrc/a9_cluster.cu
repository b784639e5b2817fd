// a9_cluster.cu -- NEXT-2: clusterizer, digits -> clusters (readings P53..P56; PAPER.md:29
// "TPC Processing (Tracking, Clustering, Compression)").  tpc_clusterize in include/tpc_track.h.
//
// Digits of a (sector,row) are cells (pad, time bin, ADC) sorted by (time, pad).  A CTA takes a row: it stages the
// row's digits as sorted 32-bit keys (time << 16 | pad) + ADC values in shared memory (rows that do not fit are read
// from global memory through the same code), and every digit finds its 8 neighbours in that sorted list: the two in
// its own time bin are its list neighbours, the three in the time bin before / after start at one binary search each.
// Peak test (P53), 3 x 3 charge-weighted centroid in integer arithmetic (P54); a peak's cluster is parked at the
// digit's index.  Then the per-row counts are scanned into the CSR row offsets, and a second pass compacts the parked
// clusters in digit order (P55).  The output arrays are the input format of tpc_track.
#include "tpc_internal.cuh"

namespace {

constexpr int A9_THREADS = 256;
constexpr int A9_SMEM_DIGITS = 12 * 1024;   // digits of one row staged in shared memory (72 KB); longer rows: global

__device__ __forceinline__ long long rdiv(long long a, long long b) {   // floor((2a + b) / (2b)), b > 0
  const long long n = 2 * a + b, d = 2 * b;
  long long q = n / d;
  if ((n % d != 0) && (n < 0)) --q;
  return q;
}

// first index in [lo, hi) whose key is >= k
__device__ __forceinline__ int lower_bound(const uint32_t* keys, int lo, int hi, uint32_t k) {
  while (lo < hi) {
    const int mid = (lo + hi) >> 1;
    if (keys[mid] < k) lo = mid + 1; else hi = mid;
  }
  return lo;
}

struct ClCfg {
  int n_rows, n_per_side, n_pads, pad_units, time_units, q_peak_min;
};

__global__ void __launch_bounds__(A9_THREADS)
a9_peaks_kernel(const ClCfg c, const uint16_t* __restrict__ pad, const uint16_t* __restrict__ time,
                const uint16_t* __restrict__ adc, const uint32_t* __restrict__ doff, uint32_t* __restrict__ g_keys,
                uint8_t* __restrict__ flag, int4* __restrict__ parked, uint32_t* __restrict__ row_count) {
  extern __shared__ uint32_t s_mem[];
  __shared__ uint32_t s_n;
  const int sr = blockIdx.x;
  const uint32_t a = doff[sr], b = doff[sr + 1];
  const int n = (int)(b - a);
  if (threadIdx.x == 0) s_n = 0;
  const bool staged = n <= A9_SMEM_DIGITS;
  uint32_t* keys = staged ? s_mem : g_keys + a;
  uint16_t* vals = (uint16_t*)(s_mem + A9_SMEM_DIGITS);
  for (int i = threadIdx.x; i < n; i += A9_THREADS) {
    keys[i] = ((uint32_t)time[a + i] << 16) | pad[a + i];
    if (staged) vals[i] = adc[a + i];
  }
  __syncthreads();
  const uint16_t* av = staged ? vals : adc + a;
  const long long y_off = ((long long)(c.n_pads - 1) * c.pad_units) / 2;
  const int side = ((sr / c.n_rows) / c.n_per_side) % 2;
  uint32_t mine = 0;
  for (int i = threadIdx.x; i < n; i += A9_THREADS) {
    const uint32_t k = keys[i];
    const int v = av[i];
    bool peak = v >= c.q_peak_min;
    if (peak) {
      long long Q = v, Sy = 0, St = 0;
      // own time bin: the list neighbours
      if (i > 0 && keys[i - 1] == k - 1u && (k & 0xffffu) != 0u) {
        const int w = av[i - 1];
        Q += w; Sy -= w;
        peak &= v > w;                       // precedes (t, p): strictly greater (P53)
      }
      if (i + 1 < n && keys[i + 1] == k + 1u) {
        const int w = av[i + 1];
        Q += w; Sy += w;
        peak &= v >= w;
      }
      // time bin before: cells (t-1, p-1), (t-1, p), (t-1, p+1)
      if ((k >> 16) != 0u) {
        const uint32_t k0 = k - 0x10000u - ((k & 0xffffu) ? 1u : 0u);   // pad 0 has no left neighbour
        int j = lower_bound(keys, 0, i, k0);
        for (; j < i && keys[j] <= k - 0x10000u + 1u; ++j) {
          const int w = av[j], dp = (int)(keys[j] & 0xffffu) - (int)(k & 0xffffu);
          Q += w; Sy += (long long)w * dp; St -= w;
          peak &= v > w;
        }
      }
      {   // time bin after
        const uint32_t k0 = k + 0x10000u - ((k & 0xffffu) ? 1u : 0u);
        int j = lower_bound(keys, i + 1, n, k0);
        for (; j < n && keys[j] <= k + 0x10000u + 1u; ++j) {
          const int w = av[j], dp = (int)(keys[j] & 0xffffu) - (int)(k & 0xffffu);
          Q += w; Sy += (long long)w * dp; St += w;
          peak &= v >= w;
        }
      }
      if (peak) {
        const long long yy = (long long)(k & 0xffffu) * c.pad_units - y_off + rdiv((long long)c.pad_units * Sy, Q);
        const long long zz = (long long)(k >> 16) * c.time_units + rdiv((long long)c.time_units * St, Q);
        parked[a + i] = make_int4((int)yy, (int)(side ? -zz : zz), (int)Q, v);
        ++mine;
      }
    }
    flag[a + i] = peak ? 1 : 0;
  }
  if (mine) atomicAdd(&s_n, mine);
  __syncthreads();
  if (threadIdx.x == 0) row_count[sr] = s_n;
}

// exclusive scan of the per-row counts into the CSR offsets (R + 1 entries); one block, chunks of 1024
__global__ void __launch_bounds__(1024)
a9_scan_kernel(int64_t R, const uint32_t* __restrict__ row_count, uint32_t* __restrict__ row_offsets,
               int32_t* __restrict__ counts, int32_t capacity) {
  __shared__ uint32_t wsum[33];
  __shared__ uint32_t s_run;
  if (threadIdx.x == 0) s_run = 0;
  __syncthreads();
  for (int64_t base = 0; base < R; base += 1024) {
    const int64_t i = base + threadIdx.x;
    const uint32_t v = i < R ? row_count[i] : 0u;
    uint32_t total;
    const uint32_t ex = block_excl_scan(v, wsum, &total);
    const uint32_t run = s_run;
    if (i < R) row_offsets[i] = run + ex;
    __syncthreads();
    if (threadIdx.x == 0) s_run = run + total;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    row_offsets[R] = s_run;
    counts[0] = (int32_t)s_run;
    counts[1] = s_run > (uint32_t)capacity ? 1 : 0;   // overflow flag: nothing beyond the capacity is written
  }
}

// compaction of the parked clusters in digit order (P55)
__global__ void __launch_bounds__(A9_THREADS)
a9_compact_kernel(const uint32_t* __restrict__ doff, const uint8_t* __restrict__ flag, const int4* __restrict__ parked,
                  const uint32_t* __restrict__ row_offsets, int32_t capacity, int32_t* __restrict__ y,
                  int32_t* __restrict__ z, int32_t* __restrict__ qtot, int32_t* __restrict__ qmax) {
  __shared__ uint32_t wsum[33];
  __shared__ uint32_t s_run;
  const int sr = blockIdx.x;
  const uint32_t a = doff[sr], b = doff[sr + 1];
  if (threadIdx.x == 0) s_run = row_offsets[sr];
  __syncthreads();
  for (uint32_t base = a; base < b; base += A9_THREADS) {
    const uint32_t i = base + threadIdx.x;
    const uint32_t f = i < b ? flag[i] : 0u;
    uint32_t total;
    const uint32_t ex = block_excl_scan(f, wsum, &total);
    const uint32_t at = s_run + ex;
    if (f && at < (uint32_t)capacity) {
      const int4 c = parked[i];
      y[at] = c.x;
      z[at] = c.y;
      qtot[at] = c.z;
      qmax[at] = c.w;
    }
    __syncthreads();
    if (threadIdx.x == 0) s_run += total;
    __syncthreads();
  }
}

}  // namespace

cudaError_t setup_a9_attributes() {
  return cudaFuncSetAttribute(a9_peaks_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, A9_SMEM_DIGITS * 6);
}

cudaError_t launch_a9_clusterize(const tpc_tracker* t, const tpc_cluster_params_t* cp, const tpc_digits_t* d,
                                 int64_t n_digits, const tpc_clusters_out_t* out, cudaStream_t st) {
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  ClCfg c;
  c.n_rows = t->g.n_rows;
  c.n_per_side = cp->n_per_side;
  c.n_pads = cp->n_pads;
  c.pad_units = cp->pad_units;
  c.time_units = cp->time_units;
  c.q_peak_min = cp->q_peak_min;
  if (R == 0) return cudaSuccess;
  (void)n_digits;
  a9_peaks_kernel<<<(unsigned)R, A9_THREADS, A9_SMEM_DIGITS * 6, st>>>(c, d->pad, d->time, d->adc, d->offsets, t->cl_keys,
                                                                      t->cl_flag, t->cl_parked, t->cl_row_count);
  a9_scan_kernel<<<1, 1024, 0, st>>>(R, t->cl_row_count, out->row_offsets, out->counts, out->capacity);
  a9_compact_kernel<<<(unsigned)R, A9_THREADS, 0, st>>>(d->offsets, t->cl_flag, t->cl_parked, out->row_offsets,
                                                        out->capacity, out->y, out->z, out->qtot, out->qmax);
  return cudaGetLastError();
}
