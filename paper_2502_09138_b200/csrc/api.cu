// api.cu -- the C ABI of libtpctrack.so (include/tpc_track.h): handle, scratch arena, stage sequencing.
// The five stages are enqueued back to back on the caller's stream; seed and track counts stay on the device
// (grids are sized by upper bounds), so a call never synchronises unless the arena has to grow.
#include <math.h>
#include <stdio.h>
#include <string.h>
#include <stdlib.h>

#include <new>

#include "tpc_internal.cuh"

namespace {

inline size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

int fail_cuda(tpc_tracker* t, cudaError_t e, const char* where) {
  t->last_err = e;
  snprintf(t->err_buf, sizeof(t->err_buf), "%s: %s", where, cudaGetErrorString(e));
  return TPC_ERR_CUDA;
}

#define TPC_CUDA(t, call)                                   \
  do {                                                      \
    cudaError_t e_ = (call);                                \
    if (e_ != cudaSuccess) return fail_cuda(t, e_, #call);  \
  } while (0)

int ceil_log2(int64_t v) {
  int s = 0;
  while (((int64_t)1 << s) < v) ++s;
  return s;
}

// Seeds a call can hold.  The worst case is n/l_min, but the per-seed scratch is ~2.2 KB and real events have far
// fewer (BASELINE configs: n/50 .. n/20), so the bound is n/16 + 4096 unless the caller reserved more; a call that
// exceeds it sets TPC_FLAG_SEED_OVERFLOW and reports the count it needs (a3, a5).
int64_t seed_capacity(const tpc_tracker* t, int64_t n) {
  const int64_t worst = n / t->params.l_min + 1;
  int64_t cap = n / 16 + 4096;
  if (cap < t->seed_reserve) cap = t->seed_reserve;
  return cap < worst ? cap : worst;
}

// Lays the scratch arrays out inside one allocation; returns the total size.  base may be NULL (size query).
size_t layout(tpc_tracker* t, char* base, int64_t n, int64_t R) {
  size_t off = 0;
  auto take = [&](size_t bytes) -> char* {
    char* p = base ? base + off : nullptr;
    off += align_up(bytes, 256);
    return p;
  };
  const int64_t s_cap = seed_capacity(t, n);
  const int64_t tiles_a3 = (n + A3_TILE - 1) / A3_TILE;
  const int64_t tiles_a5 = (s_cap + A5_TILE - 1) / A5_TILE;
  Scratch& s = t->s;
  // zeroed per call: ctl + look-back status words (kept contiguous, first in the arena)
  s.ctl = (DevCtl*)take(sizeof(DevCtl));
  s.scan_a3 = (uint64_t*)take((size_t)tiles_a3 * 8);
  s.scan_a5 = (uint64_t*)take((size_t)tiles_a5 * 8);
  s.sec_key = (uint32_t*)take((size_t)(t->g.n_sectors > 0 ? t->g.n_sectors : 1) * 4);
  s.seed_mask = (uint32_t*)take((size_t)(n / 32 + 1) * 4);
  const size_t ctl_bytes = off;
  s.srt = (int4*)take((size_t)n * 16 + 64);
  s.bin_start = (uint32_t*)take((size_t)R * t->g.nb_stride * 4);
  s.link_up = (int32_t*)take((size_t)n * 4);
  s.link_dn = (int32_t*)take((size_t)n * 4);
  s.clean_up = (int32_t*)take((size_t)n * 4);
  s.owner = (uint32_t*)take((size_t)n * 4);
  s.hit_row = (uint8_t*)take((size_t)n + 64);
  s.q_items = (uint32_t*)take((size_t)s_cap * 3 * A4_Q_BUCKETS * 4);
  s.tl_state = (int4*)take((size_t)s_cap * A4_STATE_V4 * 16);
  s.tl_span = (uint32_t*)take((size_t)s_cap * 4);
  s.seed_tmp = (int4*)take((size_t)s_cap * 16);
  s.seed_start = (int32_t*)take((size_t)s_cap * 4);
  s.seed_pos = (int32_t*)take((size_t)s_cap * 4);
  s.seed_sr = (int32_t*)take((size_t)s_cap * 4);
  s.seed_rec = (int4*)take((size_t)s_cap * 32);
  s.tl_rec = (float4*)take((size_t)s_cap * TL_REC_V4 * 16);
  s.tl_hits = (int32_t*)take((size_t)s_cap * t->g.n_rows * 4);
  s.tl_yz = (int2*)take((size_t)s_cap * ((t->g.n_rows + 3) & ~3) * 8);
  if (base) {
    t->s_cap = s_cap;
    t->tiles_a3 = tiles_a3;
    t->tiles_a5 = tiles_a5;
    t->ctl_bytes = ctl_bytes;
  }
  return off;
}

void set_grid_shape(tpc_tracker* t, int64_t y_units, int64_t z_units) {
  DevGeom& g = t->g;
  g.ny = (int)((y_units >> g.shift_y) + 1);
  g.nz = (int)((z_units >> g.shift_z) + 2);
  g.nb_stride = (int)align_up((size_t)g.ny * g.nz + 1, 4);
}

// Grid resolution of this call.  The coarsest grid (bins >= 2 x the widest search window, so a window touches at
// most 2 x 2 bins) is right while bins outnumber clusters; a dense call (pile-up: several clusters per bin) halves
// the bin sizes until bins outnumber clusters again (configs[3] literal: 36.8 -> 24.9 ms per call).  The grid only prunes, so the results do not depend on it.
void choose_grid(tpc_tracker* t, int64_t n, int64_t R) {
  DevGeom& g = t->g;
  g.shift_y = t->base_shift_y;
  g.shift_z = t->base_shift_z;
  set_grid_shape(t, t->y_units, t->z_units);
  while (R > 0 && (double)n > 1.0 * (double)R * g.ny * g.nz) {
    const int sy = g.shift_y, sz = g.shift_z;
    if (g.shift_z >= g.shift_y && g.shift_z > GRID_MIN_SHIFT) --g.shift_z;
    else if (g.shift_y > GRID_MIN_SHIFT) --g.shift_y;
    else break;
    set_grid_shape(t, t->y_units, t->z_units);
    if ((int64_t)g.ny * g.nz + 1 > GRID_MAX_BINS) {   // too many bins for a1's histogram: keep the previous shape
      g.shift_y = sy;
      g.shift_z = sz;
      set_grid_shape(t, t->y_units, t->z_units);
      break;
    }
  }
}

int ensure_arena(tpc_tracker* t, int64_t n, int64_t R) {
  if (t->arena && layout(t, nullptr, n, R) <= t->arena_bytes) {
    // same allocation, but s_cap / tile counts follow the actual n so that grids stay tight
    layout(t, (char*)t->arena, n, R);
    return TPC_OK;
  }
  int64_t cap_n = n, cap_r = R;
  if (t->arena) {   // geometric growth
    cap_n = n > t->cap_n ? n + n / 4 : t->cap_n;
    cap_r = R > t->cap_rows ? R : t->cap_rows;
    TPC_CUDA(t, cudaDeviceSynchronize());
    TPC_CUDA(t, cudaFree(t->arena));
    t->arena = nullptr;
    t->arena_bytes = 0;
  }
  const size_t bytes = layout(t, nullptr, cap_n, cap_r);
  void* p = nullptr;
  cudaError_t e = cudaMalloc(&p, bytes);
  if (e == cudaErrorMemoryAllocation) {
    cudaGetLastError();
    return TPC_ERR_NOMEM;
  }
  if (e != cudaSuccess) return fail_cuda(t, e, "cudaMalloc(arena)");
  t->arena = p;
  t->arena_bytes = bytes;
  t->cap_n = cap_n;
  t->cap_rows = cap_r;
  layout(t, (char*)p, n, R);
  return TPC_OK;
}

}  // namespace

extern "C" {
#pragma GCC visibility push(default)

void tpc_default_params(tpc_params_t* p) {
  if (!p) return;
  memset(p, 0, sizeof(*p));
  p->w_y = 1280;
  p->w_z = 1600;
  p->cost_wy = 9;
  p->cost_wz = 4;
  p->c_max = 3538944;
  p->l_min = 5;
  p->max_miss = 5;
  p->n_min_tracklet = 10;
  p->n_min_owned = 10;
  p->sigma_y = 0.1;
  p->sigma_z = 0.15;
  p->sinphi_max = 0.95;
  p->gate_d = 15.0;
  p->gate_y_cm = 2.0;
  p->gate_z_cm = 2.5;
  p->c_reset[0] = 0.25;
  p->c_reset[1] = 0.25;
  p->c_reset[2] = 0.05;
  p->c_reset[3] = 0.05;
  p->c_reset[4] = 25.0;
  p->cq_per_tesla = -0.00299792458;
}

const char* tpc_status_string(int status) {
  switch (status) {
    case TPC_OK: return "ok";
    case TPC_ERR_ARG: return "bad argument";
    case TPC_ERR_GEOMETRY: return "bad geometry (n_rows < 3, rows not ascending or extents not positive)";
    case TPC_ERR_CUDA: return "CUDA runtime error";
    case TPC_ERR_NOMEM: return "out of device memory";
    case TPC_ERR_CAPACITY: return "too many clusters for one call";
    case TPC_ERR_STATIC_SCRATCH: return "input needs more scratch than the static array of tpc_rans_encode_static holds";
    default: return "unknown status";
  }
}

const char* tpc_last_cuda_error(const tpc_tracker_t* t) { return t ? t->err_buf : ""; }

int tpc_tracker_create(const tpc_geometry_t* geo, const tpc_field_t* field, tpc_tracker_t** out) {
  if (!geo || !field || !out) return TPC_ERR_ARG;
  *out = nullptr;
  if (!geo->row_x || geo->n_sectors < 0) return TPC_ERR_ARG;
  if (geo->n_rows < 3 || !(geo->units_per_cm > 0) || !(geo->z_extent_cm > 0)) return TPC_ERR_GEOMETRY;
  if (!(geo->y_half_cm > 0) && !(geo->y_half_tan > 0)) return TPC_ERR_GEOMETRY;
  const int nr = geo->n_rows;
  // P48: rows need not be equidistant; the a2 cost weights the two gaps of a triplet by their integer pitch weights
  // nearbyint(64 * pitch / cm) (1..2^15: pitches between 1/64 cm and 512 cm).  Equal weights = P8 as written.
  bool equal_w = true;
  for (int r = 0; r + 1 < nr; ++r) {
    const double pitch = geo->row_x[r + 1] - geo->row_x[r];
    if (!(pitch > 0)) return TPC_ERR_GEOMETRY;
    const double w = nearbyint(64.0 * pitch);
    if (w < 1 || w > 32768) return TPC_ERR_GEOMETRY;
    if (w != nearbyint(64.0 * (geo->row_x[1] - geo->row_x[0]))) equal_w = false;
  }

  tpc_params_t prm;
  if (geo->params) prm = *geo->params; else tpc_default_params(&prm);
  if (prm.w_y < 0 || prm.w_z < 0 || prm.cost_wy < 0 || prm.cost_wz < 0 || prm.c_max < 0 || prm.l_min < 2 ||
      prm.max_miss < 1 || prm.n_min_tracklet < 1 || prm.n_min_tracklet > 255 || prm.n_min_owned < 1 ||
      nr > 255 || !(prm.sigma_y > 0) || !(prm.sigma_z > 0) || !(prm.sinphi_max > 0) || !(prm.sinphi_max < 1) ||
      !(prm.gate_y_cm >= 0) || !(prm.gate_z_cm >= 0))
    return TPC_ERR_ARG;
  // the a2 cost must fit int32 (equal pitches; the weighted cost is 64-bit): |ddy| <= 2 w_y, |ddz| <= 2 w_z
  {
    const double cmaxv = (double)prm.cost_wy * 4.0 * prm.w_y * prm.w_y + (double)prm.cost_wz * 4.0 * prm.w_z * prm.w_z;
    if (cmaxv >= 2147483647.0) return TPC_ERR_ARG;
  }

  tpc_tracker* t = new (std::nothrow) tpc_tracker();
  if (!t) return TPC_ERR_NOMEM;
  memset(t, 0, sizeof(*t));
  t->params = prm;
  t->bz = field->bz_tesla;
  cudaError_t e = cudaGetDevice(&t->device);
  if (e != cudaSuccess) {
    delete t;
    return TPC_ERR_CUDA;
  }

  DevGeom& g = t->g;
  g.n_sectors = geo->n_sectors;
  g.n_rows = nr;
  const int64_t gy = (int64_t)ceil(prm.gate_y_cm * geo->units_per_cm) + 2, gz = (int64_t)ceil(prm.gate_z_cm * geo->units_per_cm) + 2;
  g.shift_y = ceil_log2(2 * (prm.w_y > gy ? prm.w_y : gy) + 1);
  g.shift_z = ceil_log2(2 * (prm.w_z > gz ? prm.w_z : gz) + 1);
  const int64_t z_units = (int64_t)ceil(geo->z_extent_cm * geo->units_per_cm);
  float* dx_host = new (std::nothrow) float[nr];
  if (!dx_host) {
    delete t;
    return TPC_ERR_NOMEM;
  }
  double yh_max = 0;
  for (int r = 0; r < nr; ++r) {
    const double yh = geo->y_half_cm > 0 ? geo->y_half_cm : geo->row_x[r] * geo->y_half_tan;
    if (yh > yh_max) yh_max = yh;
  }
  const int64_t y_units = (int64_t)ceil(2.0 * yh_max * geo->units_per_cm);
  g.org_y = -(int32_t)(y_units / 2);
  for (;;) {   // coarsen until one row's histogram fits the shared memory of a CTA
    set_grid_shape(t, y_units, z_units);
    if ((int64_t)g.ny * g.nz + 1 <= GRID_MAX_BINS) break;
    if (g.nz > g.ny) ++g.shift_z; else ++g.shift_y;
  }
  t->base_shift_y = g.shift_y;
  t->base_shift_z = g.shift_z;
  t->y_units = y_units;
  t->z_units = z_units;
  for (int r = 0; r < nr; ++r) dx_host[r] = (float)(geo->row_x[r + 1 < nr ? r + 1 : r] - geo->row_x[r + 1 < nr ? r : r - 1]);
  g.w_y = prm.w_y; g.w_z = prm.w_z; g.cost_wy = prm.cost_wy; g.cost_wz = prm.cost_wz; g.c_max = prm.c_max;
  g.l_min = prm.l_min; g.max_miss = prm.max_miss; g.n_min_tracklet = prm.n_min_tracklet; g.n_min_owned = prm.n_min_owned;
  g.sy2 = (float)(prm.sigma_y * prm.sigma_y);
  g.sz2 = (float)(prm.sigma_z * prm.sigma_z);
  g.sinphi_max = (float)prm.sinphi_max;
  g.gate_d = (float)prm.gate_d;
  g.gate_y = (float)prm.gate_y_cm;
  g.gate_z = (float)prm.gate_z_cm;
  g.inv_units = (float)(1.0 / geo->units_per_cm);
  g.units = (float)geo->units_per_cm;
  g.inv_units_d = 1.0 / geo->units_per_cm;
  g.cq = (float)(prm.cq_per_tesla * field->bz_tesla);
  for (int k = 0; k < 5; ++k) g.c_reset[k] = (float)prm.c_reset[k];

  // geometry tables in one small device blob: row_x (double) | row_dx (float) | gap_w (int32)
  const size_t o_dx = align_up((size_t)nr * 8, 256);
  const size_t o_w = o_dx + align_up((size_t)nr * 4, 256);
  const size_t blob = o_w + align_up((size_t)nr * 4, 256);
  int32_t* w_host = new (std::nothrow) int32_t[nr];
  if (!w_host) {
    delete[] dx_host;
    delete t;
    return TPC_ERR_NOMEM;
  }
  for (int r = 0; r + 1 < nr; ++r) w_host[r] = (int32_t)nearbyint(64.0 * (geo->row_x[r + 1] - geo->row_x[r]));
  w_host[nr - 1] = 0;
  int rc = TPC_OK;
  e = cudaMalloc(&t->geom_blob, blob);
  if (e == cudaSuccess) e = cudaMemcpy(t->geom_blob, geo->row_x, (size_t)nr * 8, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy((char*)t->geom_blob + o_dx, dx_host, (size_t)nr * 4, cudaMemcpyHostToDevice);
  if (e == cudaSuccess) e = cudaMemcpy((char*)t->geom_blob + o_w, w_host, (size_t)nr * 4, cudaMemcpyHostToDevice);
  delete[] dx_host;
  delete[] w_host;
  g.row_x = (const double*)t->geom_blob;
  g.row_dx = (const float*)((char*)t->geom_blob + o_dx);
  g.gap_w = equal_w ? nullptr : (const int32_t*)((char*)t->geom_blob + o_w);
  if (e == cudaSuccess) e = setup_a1_attributes(t);
  if (e == cudaSuccess) e = setup_a4_attributes(t);
  if (e == cudaSuccess) e = setup_a9_attributes();
  if (e == cudaSuccess) e = setup_a2_attributes();
  for (int k = 0; k < TIMING_SETS * 6 && e == cudaSuccess; ++k) e = cudaEventCreate(&t->ev[k]);
  if (e != cudaSuccess) {
    rc = e == cudaErrorMemoryAllocation ? TPC_ERR_NOMEM : TPC_ERR_CUDA;
    cudaGetLastError();
    tpc_tracker_destroy(t);
    return rc;
  }
  *out = t;
  return TPC_OK;
}

int tpc_tracker_destroy(tpc_tracker_t* t) {
  if (!t) return TPC_ERR_ARG;
  cudaDeviceSynchronize();
  if (t->arena) cudaFree(t->arena);
  if (t->host_arena) cudaFree(t->host_arena);
  if (t->geom_blob) cudaFree(t->geom_blob);
  if (t->cl_keys) cudaFree(t->cl_keys);
  if (t->cl_flag) cudaFree(t->cl_flag);
  if (t->cl_parked) cudaFree(t->cl_parked);
  if (t->cl_row_count) cudaFree(t->cl_row_count);
  if (t->rans_scratch) cudaFree(t->rans_scratch);
  if (t->merge_sec) cudaFree(t->merge_sec);
  if (t->merge_best) cudaFree(t->merge_best);
  if (t->merge_chi2) cudaFree(t->merge_chi2);
  for (int k = 0; k < TIMING_SETS * 6; ++k)
    if (t->ev[k]) cudaEventDestroy(t->ev[k]);
  delete t;
  return TPC_OK;
}

int tpc_track(tpc_tracker_t* t, const tpc_clusters_t* cl, int64_t n, void* stream, tpc_tracks_out_t* out) {
  if (!t || !cl || !out || n < 0) return TPC_ERR_ARG;
  if (!out->counts || out->track_capacity < 0 || out->hit_capacity < 0) return TPC_ERR_ARG;
  if ((out->track_capacity > 0 && !out->tracks) || (out->hit_capacity > 0 && !out->hit_ids)) return TPC_ERR_ARG;
  if (n > 0 && (!cl->y || !cl->z)) return TPC_ERR_ARG;
  if (!cl->row_offsets) return TPC_ERR_ARG;
  if (n >= ((int64_t)1 << 31) || seed_capacity(t, n) >= 0xFFFFFF) return TPC_ERR_CAPACITY;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (n > 0 && R == 0) return TPC_ERR_ARG;   // clusters but no (sector,row) to put them in
  choose_grid(t, n, R);
  int rc = ensure_arena(t, n, R);
  if (rc != TPC_OK) return rc;
  t->last_n = n;
  t->last_ro = cl->row_offsets;
  t->last_y = cl->y;
  t->last_z = cl->z;
  TPC_CUDA(t, cudaMemsetAsync(t->s.ctl, 0, t->ctl_bytes, st));
  if (n > 0) TPC_CUDA(t, cudaMemsetAsync(t->s.owner, 0, (size_t)n * 4, st));   // a5 ownership words start empty
  cudaEvent_t* ev = t->ev + (t->timed_calls % TIMING_SETS) * 6;   // ring of event sets, one per timed call
  if (t->timing) TPC_CUDA(t, cudaEventRecord(ev[0], st));
  TPC_CUDA(t, launch_a0_check(t, cl->row_offsets, n, st));
  TPC_CUDA(t, launch_a0_origin(t, cl->z, cl->row_offsets, n, st));
  TPC_CUDA(t, launch_a1_grid(t, cl->y, cl->z, cl->row_offsets, n, st));
  if (t->timing) TPC_CUDA(t, cudaEventRecord(ev[1], st));
  TPC_CUDA(t, launch_a2_neighbours(t, cl->row_offsets, n, st));
  if (t->timing) TPC_CUDA(t, cudaEventRecord(ev[2], st));
  TPC_CUDA(t, launch_a3_seeds(t, cl->row_offsets, n, st));
  if (t->timing) TPC_CUDA(t, cudaEventRecord(ev[3], st));
  // a4 variant: large calls run the follower as four phase-specialised kernels + a vote kernel (20 % fewer
  // instructions per tracklet, but five launches and a queue tail each: measured slower below ~10 events of
  // configs[1]); small calls run the single uniform kernel.  tpc_debug_set_a4_variant overrides (tests).
  t->a4_phased = t->a4_variant ? (t->a4_variant == 2) : (n >= A4_PHASED_MIN_CLUSTERS);
  if (t->a4_phased) TPC_CUDA(t, launch_a4_phases(t, n, st));
  else TPC_CUDA(t, launch_a4_follow(t, n, st));
  if (t->timing) TPC_CUDA(t, cudaEventRecord(ev[4], st));
  TPC_CUDA(t, launch_a5_select(t, out, st));
  if (t->timing) {
    TPC_CUDA(t, cudaEventRecord(ev[5], st));
    ++t->timed_calls;
  }
  return TPC_OK;
}

int tpc_refit(tpc_tracker_t* t, const tpc_clusters_t* cl, int64_t n, void* stream, const tpc_tracks_out_t* tracks,
              tpc_track_rec_t* refit_out) {
  if (!t || !cl || !tracks || n < 0) return TPC_ERR_ARG;
  if (!tracks->counts || tracks->track_capacity < 0 || tracks->hit_capacity < 0) return TPC_ERR_ARG;
  if (tracks->track_capacity > 0 && (!tracks->tracks || !refit_out)) return TPC_ERR_ARG;
  if (tracks->hit_capacity > 0 && !tracks->hit_ids) return TPC_ERR_ARG;
  // the records of the clusters (a3) must be those of the call that produced `tracks`
  if (!t->arena || n != t->last_n || cl->row_offsets != t->last_ro || cl->y != t->last_y || cl->z != t->last_z)
    return TPC_ERR_ARG;
  TPC_CUDA(t, launch_a6_refit(t, cl->y, cl->z, tracks, refit_out, (cudaStream_t)stream));
  return TPC_OK;
}

void tpc_default_merge_params(tpc_merge_params_t* p) {
  if (!p) return;
  p->gap_max = 25;
  p->n_per_side = 18;
  p->chi2_max = 50.0;
  p->sector_angle = 20.0 * 3.14159265358979323846 / 180.0;
}

int tpc_merge(tpc_tracker_t* t, const tpc_track_rec_t* tracks, const int32_t* counts, int32_t track_capacity,
              const tpc_merge_params_t* params, void* stream, int32_t* succ, int32_t* pred, float* link_chi2,
              int32_t* merge_counts) {
  if (!t || !counts || !merge_counts || track_capacity < 0) return TPC_ERR_ARG;
  if (track_capacity > 0 && (!tracks || !succ || !pred || !link_chi2)) return TPC_ERR_ARG;
  tpc_merge_params_t mp;
  if (params) mp = *params; else tpc_default_merge_params(&mp);
  if (mp.gap_max < 1 || mp.n_per_side < 1 || !(mp.chi2_max > 0)) return TPC_ERR_ARG;
  if (track_capacity > t->merge_cap || !t->merge_sec) {
    TPC_CUDA(t, cudaDeviceSynchronize());
    if (t->merge_sec) cudaFree(t->merge_sec);
    if (t->merge_best) cudaFree(t->merge_best);
    if (t->merge_chi2) cudaFree(t->merge_chi2);
    t->merge_sec = nullptr; t->merge_best = nullptr; t->merge_chi2 = nullptr; t->merge_cap = 0;
    const size_t cap = (size_t)(track_capacity > 0 ? track_capacity : 1);
    cudaError_t e = cudaMalloc(&t->merge_sec, ((size_t)t->g.n_sectors + 2) * 4);
    if (e == cudaSuccess) e = cudaMalloc(&t->merge_best, cap * 2 * 4);
    if (e == cudaSuccess) e = cudaMalloc(&t->merge_chi2, cap * 2 * 8);
    if (e == cudaErrorMemoryAllocation) {
      cudaGetLastError();
      return TPC_ERR_NOMEM;
    }
    if (e != cudaSuccess) return fail_cuda(t, e, "cudaMalloc(merge scratch)");
    t->merge_cap = (int64_t)cap;
  }
  TPC_CUDA(t, launch_a7_merge(t, &mp, tracks, counts, track_capacity, succ, pred, link_chi2, merge_counts,
                              (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_refit_merged(tpc_tracker_t* t, const tpc_clusters_t* cl, int64_t n, void* stream, const tpc_tracks_out_t* tracks,
                     const int32_t* succ, const int32_t* pred, const tpc_merge_params_t* params,
                     tpc_track_rec_t* refit_out) {
  if (!t || !cl || !tracks || n < 0) return TPC_ERR_ARG;
  if (!tracks->counts || tracks->track_capacity < 0 || tracks->hit_capacity < 0) return TPC_ERR_ARG;
  if (tracks->track_capacity > 0 && (!tracks->tracks || !refit_out || !succ || !pred)) return TPC_ERR_ARG;
  if (tracks->hit_capacity > 0 && !tracks->hit_ids) return TPC_ERR_ARG;
  // the row list of the output hits (a5) must be that of the call that produced `tracks`
  if (!t->arena || n != t->last_n || cl->row_offsets != t->last_ro || cl->y != t->last_y || cl->z != t->last_z)
    return TPC_ERR_ARG;
  tpc_merge_params_t mp;
  if (params) mp = *params; else tpc_default_merge_params(&mp);
  if (mp.n_per_side < 1) return TPC_ERR_ARG;
  TPC_CUDA(t, launch_a6_refit_merged(t, &mp, cl->y, cl->z, tracks, succ, pred, refit_out, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_compress(tpc_tracker_t* t, const tpc_clusters_t* cl, int64_t n, void* stream, const tpc_tracks_out_t* tracks,
                 const tpc_compressed_t* out) {
  if (!t || !cl || !tracks || !out || n < 0) return TPC_ERR_ARG;
  if (!tracks->counts || tracks->track_capacity < 0 || tracks->hit_capacity < 0) return TPC_ERR_ARG;
  if (!out->hist_ry || !out->hist_rz || !out->hist_drow) return TPC_ERR_ARG;
  if (tracks->hit_capacity > 0 && (!tracks->hit_ids || !out->drow || !out->ry || !out->rz)) return TPC_ERR_ARG;
  if (tracks->track_capacity > 0 && !tracks->tracks) return TPC_ERR_ARG;
  // the row list of the output hits (a5) must be that of the call that produced `tracks`
  if (!t->arena || n != t->last_n || cl->row_offsets != t->last_ro || cl->y != t->last_y || cl->z != t->last_z)
    return TPC_ERR_ARG;
  TPC_CUDA(t, launch_a8_compress(t, cl->y, cl->z, tracks, out, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_decompress(tpc_tracker_t* t, void* stream, const tpc_tracks_out_t* tracks, const tpc_compressed_t* in,
                   int32_t* row, int32_t* y, int32_t* z) {
  if (!t || !tracks || !in || !tracks->counts || tracks->track_capacity < 0 || tracks->hit_capacity < 0) return TPC_ERR_ARG;
  if (tracks->hit_capacity > 0 && (!in->drow || !in->ry || !in->rz || !row || !y || !z)) return TPC_ERR_ARG;
  if (tracks->track_capacity > 0 && !tracks->tracks) return TPC_ERR_ARG;
  TPC_CUDA(t, launch_a8_decompress(t, tracks, in, row, y, z, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_rans_encode(tpc_tracker_t* t, const void* values, int32_t value_bytes, int64_t n, int32_t alphabet_bits,
                    int32_t chunk, void* stream, const tpc_rans_stream_t* out) {
  if (!t || !out || n < 0 || n >= ((int64_t)1 << 31) || (value_bytes != 1 && value_bytes != 4)) return TPC_ERR_ARG;
  if (alphabet_bits < 1 || alphabet_bits > 12 || chunk < 1 || chunk > 65535) return TPC_ERR_ARG;
  if (!out->freq || !out->chunk_off || !out->esc_off || !out->counts || out->payload_capacity < 0 ||
      out->escape_capacity < 0)
    return TPC_ERR_ARG;
  if (n > 0 && (!values || (out->payload_capacity > 0 && !out->payload) || (out->escape_capacity > 0 && !out->escapes)))
    return TPC_ERR_ARG;
  const size_t need = rans_scratch_bytes(n, chunk, alphabet_bits);
  if (need > t->rans_scratch_cap) {
    TPC_CUDA(t, cudaDeviceSynchronize());
    if (t->rans_scratch) cudaFree(t->rans_scratch);
    t->rans_scratch = nullptr;
    t->rans_scratch_cap = 0;
    if (cudaMalloc(&t->rans_scratch, need) != cudaSuccess) {
      cudaGetLastError();
      return TPC_ERR_NOMEM;
    }
    t->rans_scratch_cap = need;
  }
  TPC_CUDA(t, launch_a10_rans_encode(t, values, value_bytes, n, alphabet_bits, chunk, out, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_rans_decode(tpc_tracker_t* t, const tpc_rans_stream_t* in, int64_t n, int32_t alphabet_bits, int32_t chunk,
                    void* stream, void* values, int32_t value_bytes) {
  if (!t || !in || n < 0 || n >= ((int64_t)1 << 31) || (value_bytes != 1 && value_bytes != 4)) return TPC_ERR_ARG;
  if (alphabet_bits < 1 || alphabet_bits > 12 || chunk < 1 || chunk > 65535) return TPC_ERR_ARG;
  if (!in->freq || !in->chunk_off || !in->esc_off) return TPC_ERR_ARG;
  if (n > 0 && (!values || !in->payload)) return TPC_ERR_ARG;
  TPC_CUDA(t, launch_a10_rans_decode(t, in, n, alphabet_bits, chunk, values, value_bytes, (cudaStream_t)stream));
  return TPC_OK;
}

void tpc_default_cluster_params(tpc_cluster_params_t* p) {
  if (!p) return;
  p->n_pads = 223;
  p->n_per_side = 18;
  p->pad_units = 256;
  p->time_units = 330;
  p->q_peak_min = 6;
}

int tpc_clusterize(tpc_tracker_t* t, const tpc_digits_t* d, int64_t n_digits, const tpc_cluster_params_t* params,
                   void* stream, const tpc_clusters_out_t* out) {
  if (!t || !d || !out || !params || n_digits < 0 || n_digits >= ((int64_t)1 << 31)) return TPC_ERR_ARG;
  if (!d->offsets || !out->row_offsets || !out->counts || out->capacity < 0) return TPC_ERR_ARG;
  if (n_digits > 0 && (!d->pad || !d->time || !d->adc)) return TPC_ERR_ARG;
  if (out->capacity > 0 && (!out->y || !out->z || !out->qtot || !out->qmax)) return TPC_ERR_ARG;
  if (params->n_pads < 1 || params->n_pads > 32768 || params->n_per_side < 1 || params->pad_units < 1 ||
      params->time_units < 1 || params->q_peak_min < 1)
    return TPC_ERR_ARG;
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (n_digits > t->cl_cap || !t->cl_row_count) {
    TPC_CUDA(t, cudaDeviceSynchronize());
    if (t->cl_keys) cudaFree(t->cl_keys);
    if (t->cl_flag) cudaFree(t->cl_flag);
    if (t->cl_parked) cudaFree(t->cl_parked);
    if (t->cl_row_count) cudaFree(t->cl_row_count);
    t->cl_keys = nullptr; t->cl_flag = nullptr; t->cl_parked = nullptr; t->cl_row_count = nullptr; t->cl_cap = 0;
    const size_t cap = (size_t)(n_digits > 0 ? n_digits + n_digits / 8 : 1);
    cudaError_t e = cudaMalloc(&t->cl_keys, cap * 4);
    if (e == cudaSuccess) e = cudaMalloc(&t->cl_flag, cap);
    if (e == cudaSuccess) e = cudaMalloc(&t->cl_parked, cap * 16);
    if (e == cudaSuccess) e = cudaMalloc(&t->cl_row_count, (size_t)(R + 1) * 4);
    if (e == cudaErrorMemoryAllocation) {
      cudaGetLastError();
      return TPC_ERR_NOMEM;
    }
    if (e != cudaSuccess) return fail_cuda(t, e, "cudaMalloc(clusterizer scratch)");
    t->cl_cap = (int64_t)cap;
  }
  TPC_CUDA(t, launch_a9_clusterize(t, params, d, n_digits, out, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_track_host(tpc_tracker_t* t, const tpc_clusters_t* cl, int64_t n, void* stream, tpc_tracks_out_t* out) {
  if (!t || !cl || !out || n < 0) return TPC_ERR_ARG;
  if (!out->counts || out->track_capacity < 0 || out->hit_capacity < 0) return TPC_ERR_ARG;
  if ((out->track_capacity > 0 && !out->tracks) || (out->hit_capacity > 0 && !out->hit_ids)) return TPC_ERR_ARG;
  if (!cl->row_offsets || (n > 0 && (!cl->y || !cl->z))) return TPC_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  // device staging for the caller's host buffers
  size_t off = 0;
  auto take = [&](size_t bytes) { size_t o = off; off += align_up(bytes, 256); return o; };
  const size_t o_y = take((size_t)n * 4), o_z = take((size_t)n * 4), o_ro = take((size_t)(R + 1) * 4);
  const size_t o_tr = take((size_t)out->track_capacity * sizeof(tpc_track_rec_t));
  const size_t o_h = take((size_t)out->hit_capacity * 4), o_c = take(16);
  if (off > t->host_arena_bytes) {
    if (t->host_arena) {
      TPC_CUDA(t, cudaDeviceSynchronize());
      TPC_CUDA(t, cudaFree(t->host_arena));
      t->host_arena = nullptr;
      t->host_arena_bytes = 0;
    }
    cudaError_t e = cudaMalloc(&t->host_arena, off);
    if (e == cudaErrorMemoryAllocation) {
      cudaGetLastError();
      return TPC_ERR_NOMEM;
    }
    if (e != cudaSuccess) return fail_cuda(t, e, "cudaMalloc(host staging)");
    t->host_arena_bytes = off;
  }
  char* b = (char*)t->host_arena;
  tpc_clusters_t dcl = {(const int32_t*)(b + o_y), (const int32_t*)(b + o_z), (const uint32_t*)(b + o_ro)};
  tpc_tracks_out_t dout;
  dout.tracks = (tpc_track_rec_t*)(b + o_tr);
  dout.track_capacity = out->track_capacity;
  dout.hit_capacity = out->hit_capacity;
  dout.hit_ids = (int32_t*)(b + o_h);
  dout.counts = (int32_t*)(b + o_c);
  if (n > 0) {
    TPC_CUDA(t, cudaMemcpyAsync(b + o_y, cl->y, (size_t)n * 4, cudaMemcpyHostToDevice, st));
    TPC_CUDA(t, cudaMemcpyAsync(b + o_z, cl->z, (size_t)n * 4, cudaMemcpyHostToDevice, st));
  }
  TPC_CUDA(t, cudaMemcpyAsync(b + o_ro, cl->row_offsets, (size_t)(R + 1) * 4, cudaMemcpyHostToDevice, st));
  for (int attempt = 0;; ++attempt) {
    int rc = tpc_track(t, &dcl, n, stream, &dout);
    if (rc != TPC_OK) return rc;
    TPC_CUDA(t, cudaMemcpyAsync(out->counts, dout.counts, 16, cudaMemcpyDeviceToHost, st));
    TPC_CUDA(t, cudaStreamSynchronize(st));
    if (!(out->counts[2] & TPC_FLAG_SEED_OVERFLOW) || attempt == 1) break;
    t->seed_reserve = (int64_t)out->counts[3] + out->counts[3] / 8 + 1024;   // the call said what it needs: once more
  }
  const int64_t nt = out->counts[0] < out->track_capacity ? out->counts[0] : out->track_capacity;
  // a5 writes the list of every track whose hits fit below hit_capacity: copy that prefix
  const int64_t nh = out->counts[1] <= out->hit_capacity ? out->counts[1] : out->hit_capacity;
  if (nt > 0)
    TPC_CUDA(t, cudaMemcpyAsync(out->tracks, dout.tracks, (size_t)nt * sizeof(tpc_track_rec_t), cudaMemcpyDeviceToHost, st));
  if (nh > 0) TPC_CUDA(t, cudaMemcpyAsync(out->hit_ids, dout.hit_ids, (size_t)nh * 4, cudaMemcpyDeviceToHost, st));
  TPC_CUDA(t, cudaStreamSynchronize(st));
  return TPC_OK;
}

int64_t tpc_scratch_bytes(const tpc_tracker_t* t) { return t ? (int64_t)(t->arena_bytes + t->host_arena_bytes) : 0; }

int tpc_launches_per_call(const tpc_tracker_t* t) { return t ? (t->a4_phased ? 12 : 8) : 0; }

int tpc_set_concurrency(tpc_tracker_t* t, int32_t k) {
  if (!t || k < 1) return TPC_ERR_ARG;
  t->concurrency = k;
  return TPC_OK;
}

int tpc_reserve_seeds(tpc_tracker_t* t, int64_t n_seeds) {
  if (!t || n_seeds < 0) return TPC_ERR_ARG;
  if (n_seeds > t->seed_reserve) t->seed_reserve = n_seeds;
  return TPC_OK;
}

int tpc_debug_set_a2_variant(tpc_tracker_t* t, int variant) {
  if (!t || variant < 0 || variant > 1) return TPC_ERR_ARG;
  t->a2_variant = variant;
  return TPC_OK;
}

int tpc_debug_set_a4_variant(tpc_tracker_t* t, int variant) {
  if (!t || variant < 0 || variant > 2) return TPC_ERR_ARG;
  t->a4_variant = variant;
  return TPC_OK;
}

int tpc_set_stage_timing(tpc_tracker_t* t, int enable) {
  if (!t) return TPC_ERR_ARG;
  t->timing = enable != 0;
  t->timed_calls = 0;
  return TPC_OK;
}

int tpc_get_stage_ms(tpc_tracker_t* t, float ms[5]) {
  if (!t || !ms || t->timed_calls == 0) return TPC_ERR_ARG;
  cudaEvent_t* ev = t->ev + ((t->timed_calls - 1) % TIMING_SETS) * 6;
  TPC_CUDA(t, cudaEventSynchronize(ev[5]));
  for (int k = 0; k < 5; ++k) TPC_CUDA(t, cudaEventElapsedTime(&ms[k], ev[k], ev[k + 1]));
  return TPC_OK;
}

int tpc_get_stage_ms_mean(tpc_tracker_t* t, float ms[5], int32_t* n_calls) {
  if (!t || !ms || t->timed_calls == 0) return TPC_ERR_ARG;
  const int64_t m = t->timed_calls < TIMING_SETS ? t->timed_calls : TIMING_SETS;
  double acc[5] = {0, 0, 0, 0, 0};
  for (int64_t c = 0; c < m; ++c) {
    cudaEvent_t* ev = t->ev + ((t->timed_calls - 1 - c) % TIMING_SETS) * 6;
    TPC_CUDA(t, cudaEventSynchronize(ev[5]));
    for (int k = 0; k < 5; ++k) {
      float v;
      TPC_CUDA(t, cudaEventElapsedTime(&v, ev[k], ev[k + 1]));
      acc[k] += v;
    }
  }
  for (int k = 0; k < 5; ++k) ms[k] = (float)(acc[k] / (double)m);
  if (n_calls) *n_calls = (int32_t)m;
  return TPC_OK;
}

int tpc_debug_copy_links(tpc_tracker_t* t, int which, int32_t* up, int32_t* dn, void* stream) {
  if (!t || !up || !dn || (which != 0 && which != 1)) return TPC_ERR_ARG;
  if (!t->arena) return TPC_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  if (t->last_n == 0) return TPC_OK;
  TPC_CUDA(t, launch_dbg_links(t, t->last_n, which, up, dn, st));
  return TPC_OK;
}

int tpc_debug_copy_seeds(tpc_tracker_t* t, int32_t* start, int32_t* len, void* stream) {
  if (!t || !start || !len || !t->arena) return TPC_ERR_ARG;
  if (t->last_n == 0) return TPC_OK;
  TPC_CUDA(t, launch_dbg_seed_len(t, start, len, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_debug_copy_tracklets(tpc_tracker_t* t, float* par, float* cov, float* chi2, int32_t* n_hits, int32_t* hits,
                             void* stream) {
  if (!t || !t->arena) return TPC_ERR_ARG;
  if (t->last_n == 0) return TPC_OK;
  TPC_CUDA(t, launch_dbg_tracklets(t, par, cov, chi2, n_hits, hits, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_debug_copy_owner(tpc_tracker_t* t, int32_t* owner, void* stream) {
  if (!t || !owner || !t->arena) return TPC_ERR_ARG;
  if (t->last_n == 0) return TPC_OK;
  TPC_CUDA(t, launch_dbg_owner(t, t->last_n, owner, (cudaStream_t)stream));
  return TPC_OK;
}

int tpc_debug_grid_info(const tpc_tracker_t* t, int32_t* bins_stride, int32_t* nz, int32_t* shift_y, int32_t* shift_z) {
  if (!t) return TPC_ERR_ARG;
  if (bins_stride) *bins_stride = t->g.nb_stride;
  if (nz) *nz = t->g.nz;
  if (shift_y) *shift_y = t->g.shift_y;
  if (shift_z) *shift_z = t->g.shift_z;
  return TPC_OK;
}

int tpc_debug_copy_grid(tpc_tracker_t* t, int32_t* ids_sorted, uint32_t* bin_start, void* stream) {
  if (!t || !t->arena) return TPC_ERR_ARG;
  cudaStream_t st = (cudaStream_t)stream;
  const int64_t R = (int64_t)t->g.n_sectors * t->g.n_rows;
  if (ids_sorted && t->last_n > 0)
    TPC_CUDA(t, cudaMemcpy2DAsync(ids_sorted, 4, &t->s.srt->z, sizeof(int4), 4, (size_t)t->last_n,
                                  cudaMemcpyDeviceToDevice, st));
  if (bin_start && R > 0)
    TPC_CUDA(t, cudaMemcpyAsync(bin_start, t->s.bin_start, (size_t)R * t->g.nb_stride * 4, cudaMemcpyDeviceToDevice, st));
  return TPC_OK;
}

#pragma GCC visibility pop
}  // extern "C"
