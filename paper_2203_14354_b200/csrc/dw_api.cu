// dw_api.cu -- host side of the C ABI (include/darwinopt.h): context, table and geometry upload with
// validation, and the host-buffer (end-to-end) propagation entry.  No arithmetic of the method lives here.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include <stdlib.h>

#include "dw_internal.cuh"

#ifndef DW_HOST_SLOTS_DEFAULT
#define DW_HOST_SLOTS_DEFAULT 2
#endif
#ifndef DW_HOST_FIRST_DEFAULT
#define DW_HOST_FIRST_DEFAULT (1 << 20)
#endif
#ifndef DW_HOST_CHUNK_DEFAULT
#define DW_HOST_CHUNK_DEFAULT (6 << 20)
#endif

static std::string g_create_err;

int dw_fail(dw_ctx* ctx, int code, const char* fmt, ...) {
  char buf[1024];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (ctx) ctx->err = buf; else g_create_err = buf;
  return code;
}

extern "C" int dw_version(void) { return DW_VERSION; }

extern "C" const char* dw_last_error(const dw_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_err.c_str(); }

extern "C" int dw_create(int cuda_device, dw_ctx** out) {
  if (!out) return dw_fail(nullptr, DW_E_ARG, "dw_create: out is NULL");
  *out = nullptr;
  int n = 0;
  cudaError_t e = cudaGetDeviceCount(&n);
  if (e != cudaSuccess || n == 0)
    return dw_fail(nullptr, DW_E_CUDA, "dw_create: no CUDA device (%s); this library has no CPU fallback",
                   e == cudaSuccess ? "device count 0" : cudaGetErrorString(e));
  if (cuda_device < 0 || cuda_device >= n) return dw_fail(nullptr, DW_E_ARG, "dw_create: device %d of %d", cuda_device, n);
  e = cudaSetDevice(cuda_device);
  if (e != cudaSuccess) return dw_fail(nullptr, DW_E_CUDA, "cudaSetDevice: %s", cudaGetErrorString(e));
  dw_ctx* c = new dw_ctx();
  c->device = cuda_device;
  cudaDeviceGetAttribute(&c->sm_count, cudaDevAttrMultiProcessorCount, cuda_device);
  // A pool of its own for the 8-byte queue heads of the launches, which keeps its memory: the default pool gives freed memory
  // back to the system at every synchronisation (release threshold 0) and maps it again for the next launch.
  {
    cudaMemPoolProps props{};
    props.allocType = cudaMemAllocationTypePinned;
    props.handleTypes = cudaMemHandleTypeNone;
    props.location.type = cudaMemLocationTypeDevice;
    props.location.id = cuda_device;
    if (cudaMemPoolCreate(&c->pool, &props) == cudaSuccess) {
      unsigned long long keep = ~0ull;
      cudaMemPoolSetAttribute(c->pool, cudaMemPoolAttrReleaseThreshold, &keep);
    } else {
      c->pool = nullptr;
      cudaGetLastError();
    }
  }
  *out = c;
  return DW_OK;
}

static void free_geometry(dw_ctx* c) {
  cudaFree(c->d_xyz); cudaFree(c->d_idx); cudaFree(c->d_code); cudaFree(c->d_chan);
  c->d_xyz = nullptr; c->d_idx = nullptr; c->d_code = nullptr; c->d_chan = nullptr;
  dw_bvh_free(c);
  c->have_geom = false;
}

extern "C" int dw_destroy(dw_ctx* c) {
  if (!c) return DW_OK;
  cudaSetDevice(c->device);
  free_geometry(c);
  cudaFree(c->d_mat); cudaFree(c->d_surf); cudaFree(c->d_film); cudaFree(c->d_film_on);
  if (c->stage) cudaFree(c->stage);
  if (c->pool) { cudaDeviceSynchronize(); cudaMemPoolDestroy(c->pool); }
  for (int i = 0; i < dw_ctx::kStageSlotsMax; ++i) {
    if (c->stage_streams[i]) cudaStreamDestroy(c->stage_streams[i]);
    if (c->stage_events[i]) cudaEventDestroy(c->stage_events[i]);
  }
  delete c;
  return DW_OK;
}

extern "C" int dw_set_materials(dw_ctx* c, int n_mat, int nl, float l0, float dl, const float* n, const float* la,
                                const float* ls) {
  if (!c) return DW_E_ARG;
  if (n_mat < 1 || n_mat > 255 || nl < 1 || !n || !la || !ls || !(dl > 0.f) || !isfinite(l0))
    return dw_fail(c, DW_E_ARG, "dw_set_materials: bad argument (n_mat=%d n_lambda=%d dlambda=%g)", n_mat, nl, dl);
  if (c->have_geom && n_mat < c->tables.n_mat)        // the packed triangle codes index the table on the device
    return dw_fail(c, DW_E_RANGE, "dw_set_materials: geometry was validated against %d materials, got %d", c->tables.n_mat, n_mat);
  size_t m = (size_t)n_mat * nl;
  std::vector<float> h(3 * m);
  for (size_t i = 0; i < m; ++i) {
    if (!(n[i] > 0.f) || !isfinite(n[i])) return dw_fail(c, DW_E_RANGE, "dw_set_materials: refractive index [%zu] = %g", i, n[i]);
    if (!(la[i] > 0.f) || !(ls[i] > 0.f)) return dw_fail(c, DW_E_RANGE, "dw_set_materials: length [%zu] must be > 0 (or +inf)", i);
    h[i] = n[i]; h[m + i] = la[i]; h[2 * m + i] = ls[i];
  }
  DW_CUDA(c, cudaSetDevice(c->device));
  DW_CUDA(c, cudaDeviceSynchronize());
  cudaFree(c->d_mat); c->d_mat = nullptr;
  DW_CUDA(c, cudaMalloc(&c->d_mat, h.size() * sizeof(float)));
  DW_CUDA(c, cudaMemcpy(c->d_mat, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice));
  c->tables.mat = c->d_mat; c->tables.n_mat = n_mat; c->tables.nl_mat = nl;
  c->tables.mat_l0 = l0; c->tables.mat_inv_dl = 1.0f / dl;
  c->have_mat = true;
  return DW_OK;
}

extern "C" int dw_set_surfaces(dw_ctx* c, int n_surf, int nl, float l0, float dl, const float* det, const float* rd,
                               const float* rs, const float* tr) {
  if (!c) return DW_E_ARG;
  if (n_surf < 1 || n_surf > 254 || nl < 1 || !det || !rd || !rs || !tr || !(dl > 0.f) || !isfinite(l0))
    return dw_fail(c, DW_E_ARG, "dw_set_surfaces: bad argument (n_surf=%d n_lambda=%d dlambda=%g)", n_surf, nl, dl);
  if (c->have_geom && n_surf < c->tables.n_surf)
    return dw_fail(c, DW_E_RANGE, "dw_set_surfaces: geometry was validated against %d surfaces, got %d", c->tables.n_surf, n_surf);
  size_t m = (size_t)n_surf * nl;
  std::vector<float> h(4 * m);
  for (size_t i = 0; i < m; ++i) {
    float p[4] = {det[i], rd[i], rs[i], tr[i]};
    double s = 0;
    for (int k = 0; k < 4; ++k) {
      if (!(p[k] >= 0.f)) return dw_fail(c, DW_E_RANGE, "dw_set_surfaces: probability %d of entry %zu is %g", k, i, p[k]);
      s += p[k];
      h[k * m + i] = (float)s;   // cumulative
    }
    if (s > 1.0 + 1e-6) return dw_fail(c, DW_E_RANGE, "dw_set_surfaces: probabilities of entry %zu sum to %g > 1", i, s);
  }
  DW_CUDA(c, cudaSetDevice(c->device));
  DW_CUDA(c, cudaDeviceSynchronize());   // a sweep swaps tables between batches: wait for kernels reading the old ones
  cudaFree(c->d_surf); c->d_surf = nullptr;
  DW_CUDA(c, cudaMalloc(&c->d_surf, h.size() * sizeof(float)));
  DW_CUDA(c, cudaMemcpy(c->d_surf, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice));
  if (c->d_film && (n_surf != c->tables.n_surf || nl != c->tables.nl_surf || l0 != c->tables.surf_l0 || 1.0f / dl != c->tables.surf_inv_dl)) {
    cudaFree(c->d_film); cudaFree(c->d_film_on);        // films belong to the grid they were uploaded on
    c->d_film = nullptr; c->d_film_on = nullptr; c->tables.film = nullptr; c->tables.film_on = nullptr;
  }
  c->tables.surf = c->d_surf; c->tables.n_surf = n_surf; c->tables.nl_surf = nl;
  c->tables.surf_l0 = l0; c->tables.surf_inv_dl = 1.0f / dl;
  c->have_surf = true;
  return DW_OK;
}

extern "C" int dw_set_films(dw_ctx* c, int n_surf, int nl, float l0, float dl, const int32_t* film_on, const float* nf,
                            const float* kf, const float* d_nm) {
  if (!c) return DW_E_ARG;
  if (!c->have_surf) return dw_fail(c, DW_E_STATE, "dw_set_films: call dw_set_surfaces first");
  DW_CUDA(c, cudaSetDevice(c->device));
  DW_CUDA(c, cudaDeviceSynchronize());
  cudaFree(c->d_film); cudaFree(c->d_film_on);
  c->d_film = nullptr; c->d_film_on = nullptr; c->tables.film = nullptr; c->tables.film_on = nullptr;
  if (!film_on) return DW_OK;
  if (!nf || !kf || !d_nm) return dw_fail(c, DW_E_ARG, "dw_set_films: null table");
  if (n_surf != c->tables.n_surf || nl != c->tables.nl_surf || l0 != c->tables.surf_l0 || !(dl > 0.f) || 1.0f / dl != c->tables.surf_inv_dl)
    return dw_fail(c, DW_E_ARG, "dw_set_films: the grid must be the one of dw_set_surfaces (%d surfaces x %d nodes)", c->tables.n_surf, c->tables.nl_surf);
  const size_t m = (size_t)n_surf * nl;
  std::vector<float> h(3 * m);
  for (size_t i = 0; i < m; ++i) {
    if (film_on[i / nl] && (!(nf[i] > 0.f) || !(kf[i] >= 0.f) || !(d_nm[i] >= 0.f) || !isfinite(nf[i]) || !isfinite(kf[i]) || !isfinite(d_nm[i])))
      return dw_fail(c, DW_E_RANGE, "dw_set_films: entry %zu: n = %g, k = %g, thickness = %g", i, nf[i], kf[i], d_nm[i]);
    h[i] = nf[i]; h[m + i] = kf[i]; h[2 * m + i] = d_nm[i];
  }
  DW_CUDA(c, cudaMalloc(&c->d_film, h.size() * sizeof(float)));
  DW_CUDA(c, cudaMalloc(&c->d_film_on, sizeof(int32_t) * n_surf));
  DW_CUDA(c, cudaMemcpy(c->d_film, h.data(), h.size() * sizeof(float), cudaMemcpyHostToDevice));
  DW_CUDA(c, cudaMemcpy(c->d_film_on, film_on, sizeof(int32_t) * n_surf, cudaMemcpyHostToDevice));
  c->tables.film = c->d_film; c->tables.film_on = c->d_film_on;
  return DW_OK;
}

// Validation + packing of the per-triangle codes on the device (one pass, works for host and device input).
__global__ void validate_pack_kernel(int64_t n_vert, const float* __restrict__ xyz, int64_t n_tri,
                                     const int32_t* __restrict__ idx, const int32_t* __restrict__ mi,
                                     const int32_t* __restrict__ mo, const int32_t* __restrict__ sf, int n_mat,
                                     int n_surf, uint32_t* __restrict__ code, unsigned long long* __restrict__ errs) {
  int64_t t = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (t >= n_tri) return;
  int i0 = idx[3 * t], i1 = idx[3 * t + 1], i2 = idx[3 * t + 2];
  bool bad_idx = i0 < 0 || i1 < 0 || i2 < 0 || i0 >= n_vert || i1 >= n_vert || i2 >= n_vert;
  int a = mi[t], b = mo[t], s = sf[t];
  bool bad_id = a < 0 || a >= n_mat || b < 0 || b >= n_mat || s < -1 || s >= n_surf;
  if (bad_idx) { atomicAdd(&errs[0], 1ull); atomicMin(&errs[4], (unsigned long long)t); return; }
  if (bad_id) { atomicAdd(&errs[1], 1ull); atomicMin(&errs[4], (unsigned long long)t); }
  float v[9];
  bool fin = true;
  for (int k = 0; k < 3; ++k) {
    v[k] = xyz[3 * (int64_t)i0 + k]; v[3 + k] = xyz[3 * (int64_t)i1 + k]; v[6 + k] = xyz[3 * (int64_t)i2 + k];
  }
  for (int k = 0; k < 9; ++k) fin = fin && isfinite(v[k]);
  if (!fin) { atomicAdd(&errs[2], 1ull); atomicMin(&errs[4], (unsigned long long)t); return; }
  double e1x = (double)v[3] - v[0], e1y = (double)v[4] - v[1], e1z = (double)v[5] - v[2];
  double e2x = (double)v[6] - v[0], e2y = (double)v[7] - v[1], e2z = (double)v[8] - v[2];
  double cx = e1y * e2z - e1z * e2y, cy = e1z * e2x - e1x * e2z, cz = e1x * e2y - e1y * e2x;
  if (!(cx * cx + cy * cy + cz * cz > 0.0)) { atomicAdd(&errs[3], 1ull); atomicMin(&errs[4], (unsigned long long)t); }
  code[t] = (uint32_t)(a & 0xFF) | ((uint32_t)(b & 0xFF) << 8) | ((uint32_t)((s < 0 ? 0xFF : s) & 0xFF) << 16);
}

extern "C" int dw_set_geometry(dw_ctx* c, int64_t n_vert, const float* xyz, int64_t n_tri, const int32_t* idx,
                               const int32_t* mi, const int32_t* mo, const int32_t* sf, const int32_t* ch, int on_dev) {
  if (!c) return DW_E_ARG;
  if (!c->have_mat || !c->have_surf) return dw_fail(c, DW_E_STATE, "dw_set_geometry: set materials and surfaces first");
  if (n_vert < 0 || n_tri < 0 || n_tri >= (1ll << 28) || n_vert >= (1ll << 31))
    return dw_fail(c, DW_E_ARG, "dw_set_geometry: sizes out of range (n_vert=%lld n_tri=%lld)", (long long)n_vert, (long long)n_tri);
  if ((n_vert > 0 && !xyz) || (n_tri > 0 && (!idx || !mi || !mo || !sf || !ch)))
    return dw_fail(c, DW_E_ARG, "dw_set_geometry: NULL array");
  DW_CUDA(c, cudaSetDevice(c->device));
  DW_CUDA(c, cudaDeviceSynchronize());
  free_geometry(c);
  c->n_vert = n_vert; c->n_tri = n_tri;
  if (n_tri == 0) { c->have_geom = true; return DW_OK; }
  cudaMemcpyKind kind = on_dev ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
  int32_t *d_mi = nullptr, *d_mo = nullptr, *d_sf = nullptr;
  unsigned long long* d_err = nullptr;
  auto cleanup = [&]() { cudaFree(d_mi); cudaFree(d_mo); cudaFree(d_sf); cudaFree(d_err); };
#define DW_TRY(call) do { cudaError_t e__ = (call); if (e__ != cudaSuccess) { cleanup(); free_geometry(c); \
    return dw_fail(c, DW_E_CUDA, "%s failed: %s", #call, cudaGetErrorString(e__)); } } while (0)
  DW_TRY(cudaMalloc(&c->d_xyz, sizeof(float) * 3 * std::max<int64_t>(n_vert, 1)));
  DW_TRY(cudaMalloc(&c->d_idx, sizeof(int32_t) * 3 * n_tri));
  DW_TRY(cudaMalloc(&c->d_code, sizeof(uint32_t) * n_tri));
  DW_TRY(cudaMalloc(&c->d_chan, sizeof(int32_t) * n_tri));
  DW_TRY(cudaMalloc(&d_mi, sizeof(int32_t) * n_tri));
  DW_TRY(cudaMalloc(&d_mo, sizeof(int32_t) * n_tri));
  DW_TRY(cudaMalloc(&d_sf, sizeof(int32_t) * n_tri));
  DW_TRY(cudaMalloc(&d_err, sizeof(unsigned long long) * 8));
  DW_TRY(cudaMemcpy(c->d_xyz, xyz, sizeof(float) * 3 * n_vert, kind));
  DW_TRY(cudaMemcpy(c->d_idx, idx, sizeof(int32_t) * 3 * n_tri, kind));
  DW_TRY(cudaMemcpy(c->d_chan, ch, sizeof(int32_t) * n_tri, kind));
  DW_TRY(cudaMemcpy(d_mi, mi, sizeof(int32_t) * n_tri, kind));
  DW_TRY(cudaMemcpy(d_mo, mo, sizeof(int32_t) * n_tri, kind));
  DW_TRY(cudaMemcpy(d_sf, sf, sizeof(int32_t) * n_tri, kind));
  unsigned long long h_err[8] = {0, 0, 0, 0, ~0ull, 0, 0, 0};
  DW_TRY(cudaMemcpy(d_err, h_err, sizeof h_err, cudaMemcpyHostToDevice));
  validate_pack_kernel<<<(unsigned)((n_tri + 255) / 256), 256>>>(n_vert, c->d_xyz, n_tri, c->d_idx, d_mi, d_mo, d_sf,
                                                                 c->tables.n_mat, c->tables.n_surf, c->d_code, d_err);
  DW_TRY(cudaGetLastError());
  DW_TRY(cudaMemcpy(h_err, d_err, sizeof h_err, cudaMemcpyDeviceToHost));
#undef DW_TRY
  cleanup();
  if (h_err[0] || h_err[1] || h_err[2] || h_err[3]) {
    free_geometry(c);
    return dw_fail(c, DW_E_RANGE,
                   "dw_set_geometry: %llu triangles with vertex index out of range, %llu with material/surface id out of "
                   "range, %llu with non-finite vertices, %llu with zero area (first bad triangle %llu)",
                   h_err[0], h_err[1], h_err[2], h_err[3], h_err[4]);
  }
  c->have_geom = true;
  // Grow the context's pool now to what a build of this geometry takes (about 400 bytes per reference, 1.3 references per triangle
  // on the paper's meshes), so that mapping the memory is part of the upload and not of the first dw_build_bvh; the pool keeps it.
  if (c->pool) {
    void* warm = nullptr;
    if (cudaMallocFromPoolAsync(&warm, 600 * (size_t)n_tri + (8u << 20), c->pool, nullptr) == cudaSuccess) {
      cudaFreeAsync(warm, nullptr);
      cudaStreamSynchronize(nullptr);
    } else {
      cudaGetLastError();
    }
  }
  return DW_OK;
}

extern "C" int dw_build_bvh(dw_ctx* c, const dw_build_params* p, dw_build_stats* st, void* stream) {
  if (!c) return DW_E_ARG;
  if (!c->have_geom) return dw_fail(c, DW_E_STATE, "dw_build_bvh: no geometry");
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_bvh_build_impl(c, p, st, (cudaStream_t)stream);
}

extern "C" int dw_refit_bvh(dw_ctx* c, int64_t n_vert, const float* xyz, int on_dev, dw_refit_stats* st, void* stream) {
  if (!c) return DW_E_ARG;
  if (!c->built || !c->have_geom) return dw_fail(c, DW_E_STATE, "dw_refit_bvh: build the BVH first");
  if (n_vert != c->n_vert) return dw_fail(c, DW_E_ARG, "dw_refit_bvh: %lld vertices, the geometry has %lld", (long long)n_vert, (long long)c->n_vert);
  if (n_vert > 0 && !xyz) return dw_fail(c, DW_E_ARG, "dw_refit_bvh: NULL array");
  DW_CUDA(c, cudaSetDevice(c->device));
  DW_CUDA(c, cudaDeviceSynchronize());                           // no query of the old tree may still be running
  return dw_bvh_refit_impl(c, xyz, on_dev, st, (cudaStream_t)stream);
}

extern "C" int dw_first_hit(dw_ctx* c, int64_t n, const float* ox, const float* oy, const float* oz, const float* dx,
                            const float* dy, const float* dz, const int32_t* ex, int32_t* tri, float* dist, void* stream) {
  if (!c) return DW_E_ARG;
  if (!c->built) return dw_fail(c, DW_E_STATE, "dw_first_hit: build the BVH first");
  if (n < 0 || (n > 0 && (!ox || !oy || !oz || !dx || !dy || !dz || !tri || !dist)))
    return dw_fail(c, DW_E_ARG, "dw_first_hit: bad argument");
  if (n == 0) return DW_OK;
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_first_hit_impl(c, n, ox, oy, oz, dx, dy, dz, ex, tri, dist, (cudaStream_t)stream);
}

extern "C" int dw_render(dw_ctx* c, const dw_camera* cam, int32_t* tri, float* depth, uint8_t* shade, void* stream) {
  if (!c) return DW_E_ARG;
  if (!c->built) return dw_fail(c, DW_E_STATE, "dw_render: build the BVH first");
  if (!cam) return dw_fail(c, DW_E_ARG, "dw_render: NULL camera");
  if (cam->width < 1 || cam->height < 1 || cam->width > 32768 || cam->height > 32768)
    return dw_fail(c, DW_E_ARG, "dw_render: image size %d x %d out of range (1..32768)", cam->width, cam->height);
  if (!(cam->fov_y_deg > 0.f && cam->fov_y_deg < 180.f)) return dw_fail(c, DW_E_ARG, "dw_render: fov_y_deg must be in (0, 180)");
  for (int a = 0; a < 3; ++a)
    if (!isfinite(cam->eye[a])) return dw_fail(c, DW_E_ARG, "dw_render: eye must be finite");
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_render_impl(c, cam, tri, depth, shade, (cudaStream_t)stream);
}

static int check_batch(dw_ctx* c, const char* who, const dw_photons* in, int32_t max_steps, const dw_hists* h) {
  if (!c->built) return dw_fail(c, DW_E_STATE, "%s: build the BVH first", who);
  if (!in || in->n < 0 || max_steps < 0) return dw_fail(c, DW_E_ARG, "%s: bad batch / max_steps", who);
  if (in->n > 0 && (!in->px || !in->py || !in->pz || !in->kx || !in->ky || !in->kz || !in->ex || !in->ey || !in->ez ||
                    !in->wavelength || !in->t0))
    return dw_fail(c, DW_E_ARG, "%s: NULL photon array", who);
  if (h) {
    if (h->n_chan < 0 || h->n_bins < 0 || (h->chan_count && h->n_chan == 0 && false))
      return dw_fail(c, DW_E_ARG, "%s: bad histogram sizes", who);
    if (h->time_hist && h->n_bins > 0 && !(h->dt > 0.f)) return dw_fail(c, DW_E_ARG, "%s: time histogram needs dt > 0", who);
  }
  return DW_OK;
}

extern "C" int dw_propagate(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_results* out,
                            const dw_hists* hist, const dw_propagate_params* params, void* stream) {
  if (!c) return DW_E_ARG;
  int rc = check_batch(c, "dw_propagate", in, max_steps, hist);
  if (rc) return rc;
  if (in->n == 0) return DW_OK;
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_propagate_impl(c, in, seed, max_steps, out, hist, params, (cudaStream_t)stream);
}

extern "C" int dw_propagate_counters(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_propagate_params* params,
                                     uint64_t* out) {
  if (!c) return DW_E_ARG;
  if (!out) return dw_fail(c, DW_E_ARG, "dw_propagate_counters: counters_out is NULL");
  int rc = check_batch(c, "dw_propagate_counters", in, max_steps, nullptr);
  if (rc) return rc;
  for (int i = 0; i < DW_N_COUNTERS; ++i) out[i] = 0;
  if (in->n == 0) return DW_OK;
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_propagate_counters_impl(c, in, seed, max_steps, params, out, DW_N_COUNTERS);
}

// Counting over the per-photon results (dw_tally).  Neighbouring photons share their source, so equal keys are merged inside the
// warp first (__match_any_sync) and each distinct key costs one atomic.
__device__ __forceinline__ void warp_count64(unsigned long long* base, long long key, bool on) {
  const int lane = threadIdx.x & 31;
  unsigned peers = __match_any_sync(0xffffffffu, on ? key : (long long)(-1 - lane));
  if (on && lane == (__ffs(peers) - 1)) atomicAdd(base + key, (unsigned long long)__popc(peers));
}
__device__ __forceinline__ void warp_count32(unsigned* base, long long key, bool on) {
  const int lane = threadIdx.x & 31;
  unsigned peers = __match_any_sync(0xffffffffu, on ? key : (long long)(-1 - lane));
  if (on && lane == (__ffs(peers) - 1)) atomicAdd(base + key, (unsigned)__popc(peers));
}
__global__ void tally_kernel(dw_results R, int64_t n, int64_t pps, dw_tally_tables T) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  const bool live = i < n;
  const int64_t s = live ? i / pps : 0;
  const uint32_t fate = live ? (R.flags[i] & 0xFu) : 0xFu;
  if (T.fate_by_source) warp_count64((unsigned long long*)T.fate_by_source, s * 8 + (fate & 7u), live);
  const bool det = live && fate == DW_FATE_DETECTED;
  if (T.detected && R.channel && T.channel_group) {
    int g = -1;
    if (det) { const int c = R.channel[i]; if (c >= 0 && c < T.n_chan) g = T.channel_group[c]; }
    warp_count64((unsigned long long*)T.detected, s * T.n_groups + g, det && g >= 0 && g < T.n_groups);
  }
  if (T.time_hist && R.t && T.n_bins > 0) {
    long long b = 0;
    if (det) {
      const float fb = floorf((R.t[i] - T.t_min) / T.dt);
      b = fb < 0.f ? 0 : (fb > (float)(T.n_bins - 1) ? T.n_bins - 1 : (long long)fb);
    }
    warp_count32(T.time_hist, s * T.n_bins + b, det);
  }
  if (T.absorbed_by_component && R.last_tri && T.tri_component) {
    int k = -1;
    if (live && fate == DW_FATE_SURFACE_ABSORBED) { const int t = R.last_tri[i]; if (t >= 0 && t < T.n_tri_map) k = T.tri_component[t]; }
    warp_count64((unsigned long long*)T.absorbed_by_component, k, k >= 0 && k < T.n_components);
  }
}

extern "C" int dw_tally(dw_ctx* c, const dw_results* res, int64_t n, int64_t pps, const dw_tally_tables* T, void* stream) {
  if (!c) return DW_E_ARG;
  if (!res || !T || n < 0 || pps < 1) return dw_fail(c, DW_E_ARG, "dw_tally: null argument, n < 0 or photons_per_source < 1");
  if (n == 0) return DW_OK;
  if (!res->flags) return dw_fail(c, DW_E_ARG, "dw_tally: results->flags is required");
  if ((T->detected && (T->n_groups < 1 || T->n_chan < 0)) || (T->absorbed_by_component && (T->n_components < 1 || T->n_tri_map < 0)) ||
      (T->time_hist && T->n_bins > 0 && !(T->dt > 0.f)))
    return dw_fail(c, DW_E_ARG, "dw_tally: n_groups / n_components must be >= 1 and dt > 0 for the tables that are asked for");
  DW_CUDA(c, cudaSetDevice(c->device));
  tally_kernel<<<(unsigned)((n + 255) / 256), 256, 0, (cudaStream_t)stream>>>(*res, n, pps, *T);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}

// LCE and t90 from the accumulated tables (dw_tally_finish).  One warp per source: the row of the arrival-time
// histogram is summed, then scanned 32 bins at a time until the running count reaches quantile x total; the crossing is placed
// linearly inside that bin.  Sums and divisions in double (the counts are integers), one rounding to fp32 at the end.
__global__ void tally_finish_kernel(dw_tally_tables T, int64_t ns, double quantile, float* __restrict__ lce, float* __restrict__ t90) {
  const int lane = threadIdx.x & 31;
  const int64_t s = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  if (s >= ns) return;
  if (lce) {
    unsigned long long gen = lane < 8 ? (unsigned long long)T.fate_by_source[s * 8 + lane] : 0ull;
    for (int o = 4; o > 0; o >>= 1) gen += __shfl_xor_sync(0xffffffffu, gen, o);
    gen = __shfl_sync(0xffffffffu, gen, 0);
    for (int g = lane; g < T.n_groups; g += 32)
      lce[s * T.n_groups + g] = gen ? (float)((double)T.detected[s * T.n_groups + g] / (double)gen) : __int_as_float(0x7fc00000);
  }
  if (t90) {
    const uint32_t* row = T.time_hist + s * T.n_bins;
    unsigned long long tot = 0;
    for (int64_t b = lane; b < T.n_bins; b += 32) tot += row[b];
    for (int o = 16; o > 0; o >>= 1) tot += __shfl_xor_sync(0xffffffffu, tot, o);
    float res = __int_as_float(0x7fc00000);                     // NaN: nothing was detected
    if (tot > 0) {
      const double target = quantile * (double)tot;
      unsigned long long before = 0;                            // count of all bins below the current group of 32
      for (int64_t b0 = 0; b0 < T.n_bins; b0 += 32) {
        const int64_t b = b0 + lane;
        const unsigned long long mine = b < T.n_bins ? row[b] : 0u;
        unsigned long long incl = mine;                         // inclusive prefix sum over the group
        for (int o = 1; o < 32; o <<= 1) {
          const unsigned long long up = __shfl_up_sync(0xffffffffu, incl, o);
          if (lane >= o) incl += up;
        }
        const unsigned hit = __ballot_sync(0xffffffffu, b < T.n_bins && (double)(before + incl) >= target && mine > 0);
        if (hit) {
          const int l = __ffs(hit) - 1;
          const unsigned long long below = before + __shfl_sync(0xffffffffu, incl, l) - __shfl_sync(0xffffffffu, mine, l);
          const double inside = (target - (double)below) / (double)__shfl_sync(0xffffffffu, mine, l);
          res = (float)((double)T.t_min + (double)T.dt * ((double)(b0 + l) + inside));
          break;
        }
        before += __shfl_sync(0xffffffffu, incl, 31);
      }
    }
    if (lane == 0) t90[s] = res;
  }
}

extern "C" int dw_tally_finish(dw_ctx* c, const dw_tally_tables* T, int64_t ns, float quantile, float* lce, float* t90, void* stream) {
  if (!c) return DW_E_ARG;
  if (!T || ns < 0 || !(quantile > 0.f && quantile <= 1.f)) return dw_fail(c, DW_E_ARG, "dw_tally_finish: null tables, n_sources < 0 or quantile outside (0, 1]");
  if (lce && (!T->detected || !T->fate_by_source || T->n_groups < 1)) return dw_fail(c, DW_E_ARG, "dw_tally_finish: lce_out needs detected, fate_by_source and n_groups >= 1");
  if (t90 && (!T->time_hist || T->n_bins < 1 || !(T->dt > 0.f))) return dw_fail(c, DW_E_ARG, "dw_tally_finish: t90_out needs time_hist, n_bins >= 1 and dt > 0");
  if (ns == 0 || (!lce && !t90)) return DW_OK;
  DW_CUDA(c, cudaSetDevice(c->device));
  tally_finish_kernel<<<(unsigned)((ns * 32 + 255) / 256), 256, 0, (cudaStream_t)stream>>>(*T, ns, (double)quantile, lce, t90);
  DW_CUDA(c, cudaGetLastError());
  return DW_OK;
}

static int check_source(dw_ctx* c, const char* who, const dw_source* src) {
  if (src->shape < DW_SOURCE_POINT || src->shape > DW_SOURCE_BALL) return dw_fail(c, DW_E_ARG, "%s: unknown shape %d", who, src->shape);
  const float chk[] = {src->centre[0], src->centre[1], src->centre[2], src->radius, src->z0, src->z1, src->lambda_mean, src->lambda_sigma,
                       src->t_start, src->tau1, src->tau3, src->f_singlet};
  for (float v : chk) if (!std::isfinite(v)) return dw_fail(c, DW_E_ARG, "%s: non-finite source parameter", who);
  if (src->radius < 0.f || src->lambda_sigma < 0.f || src->tau1 < 0.f || src->tau3 < 0.f || src->z1 < src->z0 ||
      src->f_singlet < 0.f || src->f_singlet > 1.f)
    return dw_fail(c, DW_E_ARG, "%s: radius, sigma, tau must be >= 0, z0 <= z1, 0 <= f_singlet <= 1", who);
  return DW_OK;
}
int dw_check_source(dw_ctx* c, const char* who, const dw_source* src) { return check_source(c, who, src); }   // for dw_static.cu
static int check_emit_out(dw_ctx* c, const char* who, const dw_photons* out) {
  if (out->n < 0) return dw_fail(c, DW_E_ARG, "%s: n < 0", who);
  const float* const arr[11] = {out->px, out->py, out->pz, out->kx, out->ky, out->kz, out->ex, out->ey, out->ez, out->wavelength, out->t0};
  if (out->n > 0) for (const float* a : arr) if (!a) return dw_fail(c, DW_E_ARG, "%s: null output array", who);
  return DW_OK;
}

extern "C" int dw_emit(dw_ctx* c, const dw_source* src, uint64_t seed, const dw_photons* out, void* stream) {
  if (!c) return DW_E_ARG;
  if (!src || !out) return dw_fail(c, DW_E_ARG, "dw_emit: null source or output");
  int rc = check_emit_out(c, "dw_emit", out);
  if (rc) return rc;
  rc = check_source(c, "dw_emit", src);
  if (rc) return rc;
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_emit_impl(c, src, seed, out, (cudaStream_t)stream);
}

// Stream-ordered scratch from the context's pool (memory is kept between calls).
static cudaError_t scratch_alloc(dw_ctx* c, void** p, size_t bytes, cudaStream_t s) {
  return c->pool ? cudaMallocFromPoolAsync(p, bytes, c->pool, s) : cudaMallocAsync(p, bytes, s);
}

static int upload_sources(dw_ctx* c, const char* who, const dw_source* sources, int64_t ns, dw_source** d_out, cudaStream_t s) {
  for (int64_t i = 0; i < ns; ++i) { int rc = check_source(c, who, sources + i); if (rc) return rc; }
  DW_CUDA(c, scratch_alloc(c, (void**)d_out, sizeof(dw_source) * (size_t)ns, s));
  cudaError_t e = cudaMemcpyAsync(*d_out, sources, sizeof(dw_source) * (size_t)ns, cudaMemcpyHostToDevice, s);
  if (e != cudaSuccess) { cudaFreeAsync(*d_out, s); *d_out = nullptr; return dw_fail(c, DW_E_CUDA, "%s: copy of the sources failed: %s", who, cudaGetErrorString(e)); }
  return DW_OK;
}

extern "C" int dw_emit_sources(dw_ctx* c, const dw_source* sources, int64_t ns, int64_t pps, uint64_t seed, const dw_photons* out, void* stream) {
  if (!c) return DW_E_ARG;
  if (!sources || !out || ns < 1 || pps < 1) return dw_fail(c, DW_E_ARG, "dw_emit_sources: null argument, n_sources < 1 or photons_per_source < 1");
  int rc = check_emit_out(c, "dw_emit_sources", out);
  if (rc) return rc;
  if (out->n > ns * pps) return dw_fail(c, DW_E_ARG, "dw_emit_sources: %lld photons need more than %lld sources of %lld", (long long)out->n, (long long)ns, (long long)pps);
  if (out->n == 0) return DW_OK;
  DW_CUDA(c, cudaSetDevice(c->device));
  cudaStream_t s = (cudaStream_t)stream;
  dw_source* d_src = nullptr;
  rc = upload_sources(c, "dw_emit_sources", sources, ns, &d_src, s);
  if (rc) return rc;
  rc = dw_emit_sources_impl(c, d_src, pps, seed, out, s);
  cudaFreeAsync(d_src, s);
  return rc;
}

extern "C" int dw_design_study(dw_ctx* c, const dw_source* sources, int64_t ns, int64_t pps, uint64_t seed, int32_t max_steps,
                               const dw_tally_tables* T, int64_t spb, float quantile, float* lce, float* t90, void* stream) {
  if (!c) return DW_E_ARG;
  if (!c->built) return dw_fail(c, DW_E_STATE, "dw_design_study: build the BVH first");
  if (!sources || !T || ns < 1 || pps < 1 || max_steps < 0) return dw_fail(c, DW_E_ARG, "dw_design_study: null argument, n_sources < 1, photons_per_source < 1 or max_steps < 0");
  if (pps > (int64_t(1) << 30)) return dw_fail(c, DW_E_ARG, "dw_design_study: photons_per_source above 2^30");
  if (spb <= 0) spb = std::max<int64_t>(1, (int64_t(1) << 25) / pps);
  spb = std::min(spb, ns);
  DW_CUDA(c, cudaSetDevice(c->device));
  cudaStream_t s = (cudaStream_t)stream;
  dw_source* d_src = nullptr;
  int rc = upload_sources(c, "dw_design_study", sources, ns, &d_src, s);
  if (rc) return rc;
  const int64_t cap = spb * pps;                       // photons of a full batch
  float* buf = nullptr;                                // 11 input arrays + flags, channel, t, last_tri
  cudaError_t e = scratch_alloc(c, (void**)&buf, sizeof(float) * 15 * (size_t)cap, s);
  if (e != cudaSuccess) { cudaFreeAsync(d_src, s); return dw_fail(c, DW_E_CUDA, "dw_design_study: %zu bytes of batch buffers: %s", sizeof(float) * 15 * (size_t)cap, cudaGetErrorString(e)); }
  auto arr = [&](int k) { return buf + (size_t)k * cap; };
  for (int64_t s0 = 0; s0 < ns && rc == DW_OK; s0 += spb) {
    const int64_t nsb = std::min(spb, ns - s0), nb = nsb * pps;
    dw_photons ph{nb, (uint64_t)(s0 * pps), arr(0), arr(1), arr(2), arr(3), arr(4), arr(5), arr(6), arr(7), arr(8), arr(9), arr(10)};
    dw_results res{};
    res.flags = (uint32_t*)arr(11); res.channel = (int32_t*)arr(12); res.t = arr(13); res.last_tri = (int32_t*)arr(14);
    dw_tally_tables tb = *T;                           // the same tables seen from source s0 on
    if (tb.detected) tb.detected += s0 * tb.n_groups;
    if (tb.time_hist) tb.time_hist += s0 * tb.n_bins;
    if (tb.fate_by_source) tb.fate_by_source += s0 * 8;
    rc = dw_emit_sources_impl(c, d_src + s0, pps, seed, &ph, s);
    if (rc == DW_OK) rc = dw_propagate_impl(c, &ph, seed, max_steps, &res, nullptr, nullptr, s);
    if (rc == DW_OK) rc = dw_tally(c, &res, nb, pps, &tb, s);
  }
  if (rc == DW_OK && (lce || t90)) rc = dw_tally_finish(c, T, ns, quantile, lce, t90, s);
  cudaFreeAsync(buf, s);
  cudaFreeAsync(d_src, s);
  return rc;
}

extern "C" int dw_debug_philox(dw_ctx* c, uint64_t seed, uint64_t base, uint32_t step, uint32_t block, int64_t n,
                               uint32_t* out_raw, float* out_u, void* stream) {
  if (!c) return DW_E_ARG;
  if (n < 0) return dw_fail(c, DW_E_ARG, "dw_debug_philox: n < 0");
  if (n == 0) return DW_OK;
  DW_CUDA(c, cudaSetDevice(c->device));
  return dw_debug_philox_impl(c, seed, base, step, block, n, out_raw, out_u, (cudaStream_t)stream);
}

extern "C" int dw_last_launch(const dw_ctx* c, int32_t* grid, int32_t* block, int32_t* smem, int64_t* n_launches) {
  if (!c) return DW_E_ARG;
  if (grid) *grid = c->last_grid;
  if (block) *block = c->last_block;
  if (smem) *smem = c->last_smem;
  if (n_launches) *n_launches = c->n_launches;
  return DW_OK;
}

// ---------------------------------------------------------------------------------------------------------
// Host-buffer entry: chunks of the batch are copied to a device staging area on two alternating streams so
// that the copy of chunk i+1 overlaps the propagation of chunk i; results are copied back per chunk and the
// reductions are added into the host arrays at the end.
// ---------------------------------------------------------------------------------------------------------
namespace {
struct StageLayout {
  int64_t chunk;
  size_t in_off[11], out_off[14], hist_off[4], total;
};
inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }
}  // namespace

extern "C" int dw_propagate_host(dw_ctx* c, const dw_photons* in, uint64_t seed, int32_t max_steps,
                                 const dw_results* out, const dw_hists* hist, const dw_propagate_params* params) {
  if (!c) return DW_E_ARG;
  int rc = check_batch(c, "dw_propagate_host", in, max_steps, hist);
  if (rc) return rc;
  DW_CUDA(c, cudaSetDevice(c->device));
  const int64_t n = in->n;
  if (n == 0) return DW_OK;
  // photons per staged chunk: DW_HOST_CHUNK in the environment overrides the default (a tuning knob for the end-to-end path)
  int64_t chunk_max = DW_HOST_CHUNK_DEFAULT;
  if (const char* ev = getenv("DW_HOST_CHUNK")) { long long v = atoll(ev); if (v >= 1024) chunk_max = v; }
  const int64_t chunk = std::min<int64_t>(n, chunk_max);
  // staging slots (= streams = chunks in flight): DW_HOST_SLOTS in the environment, 2..4
  int n_slots = DW_HOST_SLOTS_DEFAULT;
  if (const char* ev = getenv("DW_HOST_SLOTS")) { int v = atoi(ev); if (v >= 2 && v <= dw_ctx::kStageSlotsMax) n_slots = v; }
  const int64_t n_chan = hist ? hist->n_chan : 0, n_bins = hist ? hist->n_bins : 0;
  // layout: n_slots x (11 inputs + up to 14 outputs) + histograms
  size_t per_slot = 25 * align256(sizeof(float) * chunk);
  size_t hist_bytes = align256(8 * n_chan) + align256(4 * n_bins) + align256(64) + align256(8);
  size_t need = n_slots * per_slot + hist_bytes;
  if (c->stage_bytes < need) {
    if (c->stage) cudaFree(c->stage);
    c->stage = nullptr; c->stage_bytes = 0;
    DW_CUDA(c, cudaMalloc(&c->stage, need));
    c->stage_bytes = need;
  }
  for (int i = 0; i < n_slots; ++i) {
    if (!c->stage_streams[i]) DW_CUDA(c, cudaStreamCreateWithFlags(&c->stage_streams[i], cudaStreamNonBlocking));
    if (!c->stage_events[i]) DW_CUDA(c, cudaEventCreateWithFlags(&c->stage_events[i], cudaEventDisableTiming));
  }
  char* base = (char*)c->stage;
  char* hbase = base + n_slots * per_slot;
  uint64_t* d_chan = (uint64_t*)hbase;
  uint32_t* d_time = (uint32_t*)(hbase + align256(8 * n_chan));
  uint64_t* d_fate = (uint64_t*)(hbase + align256(8 * n_chan) + align256(4 * n_bins));
  uint64_t* d_steps = (uint64_t*)(hbase + align256(8 * n_chan) + align256(4 * n_bins) + align256(64));
  DW_CUDA(c, cudaMemsetAsync(hbase, 0, hist_bytes, c->stage_streams[0]));
  DW_CUDA(c, cudaEventRecord(c->stage_events[0], c->stage_streams[0]));
  for (int i = 1; i < n_slots; ++i) DW_CUDA(c, cudaStreamWaitEvent(c->stage_streams[i], c->stage_events[0], 0));
  const float* src[11] = {in->px, in->py, in->pz, in->kx, in->ky, in->kz, in->ex, in->ey, in->ez, in->wavelength, in->t0};
  void* dst_host[14] = {nullptr};
  if (out) {
    void* tmp[14] = {out->flags, out->channel, out->t, out->steps, out->last_tri, out->x, out->y, out->z,
                     out->kx, out->ky, out->kz, out->ex, out->ey, out->ez};
    memcpy(dst_host, tmp, sizeof tmp);
  }
  // Chunks grow: a small first one so that the device starts after a short copy, then three times larger each time up to `chunk`
  // (every chunk is its own launch with its own tail, so few large chunks are better once the pipeline is running).
  int64_t first = std::min<int64_t>(chunk, DW_HOST_FIRST_DEFAULT);
  if (const char* ev = getenv("DW_HOST_FIRST")) { long long v = atoll(ev); if (v >= 1024) first = std::min<int64_t>(chunk, v); }
  int slot = 0;
  int64_t m_next = first;
  for (int64_t a = 0, m = 0; a < n; a += m, slot = (slot + 1) % n_slots) {
    m = std::min<int64_t>(m_next, n - a);
    m_next = std::min<int64_t>(chunk, 3 * m_next);
    cudaStream_t s = c->stage_streams[slot];
    char* sb = base + slot * per_slot;
    float* din[11];
    for (int k = 0; k < 11; ++k) {
      din[k] = (float*)(sb + k * align256(sizeof(float) * chunk));
      DW_CUDA(c, cudaMemcpyAsync(din[k], src[k] + a, sizeof(float) * m, cudaMemcpyHostToDevice, s));
    }
    void* dout[14];
    for (int k = 0; k < 14; ++k) dout[k] = dst_host[k] ? (void*)(sb + (11 + k) * align256(sizeof(float) * chunk)) : nullptr;
    dw_photons pin{m, in->photon_id_base + (uint64_t)a, din[0], din[1], din[2], din[3], din[4], din[5], din[6], din[7], din[8], din[9], din[10]};
    dw_results pout{(uint32_t*)dout[0], (int32_t*)dout[1], (float*)dout[2], (uint32_t*)dout[3], (int32_t*)dout[4],
                    (float*)dout[5], (float*)dout[6], (float*)dout[7], (float*)dout[8], (float*)dout[9], (float*)dout[10],
                    (float*)dout[11], (float*)dout[12], (float*)dout[13]};
    dw_hists ph{n_chan, (hist && hist->chan_count) ? d_chan : nullptr, n_bins, hist ? hist->t_min : 0.f, hist ? hist->dt : 1.f,
                (hist && hist->time_hist) ? d_time : nullptr, (hist && hist->fate_count) ? d_fate : nullptr,
                (hist && hist->total_steps) ? d_steps : nullptr};
    rc = dw_propagate_impl(c, &pin, seed, max_steps, &pout, hist ? &ph : nullptr, params, s);
    if (rc) return rc;
    for (int k = 0; k < 14; ++k)
      if (dst_host[k]) DW_CUDA(c, cudaMemcpyAsync((char*)dst_host[k] + 4 * a, dout[k], 4 * m, cudaMemcpyDeviceToHost, s));
  }
  for (int i = 0; i < n_slots; ++i) DW_CUDA(c, cudaStreamSynchronize(c->stage_streams[i]));
  if (hist) {
    std::vector<uint64_t> hc((size_t)n_chan), hf(8), hs(1);
    std::vector<uint32_t> ht((size_t)n_bins);
    if (hist->chan_count && n_chan) {
      DW_CUDA(c, cudaMemcpy(hc.data(), d_chan, 8 * n_chan, cudaMemcpyDeviceToHost));
      for (int64_t i = 0; i < n_chan; ++i) hist->chan_count[i] += hc[i];
    }
    if (hist->time_hist && n_bins) {
      DW_CUDA(c, cudaMemcpy(ht.data(), d_time, 4 * n_bins, cudaMemcpyDeviceToHost));
      for (int64_t i = 0; i < n_bins; ++i) hist->time_hist[i] += ht[i];
    }
    if (hist->fate_count) {
      DW_CUDA(c, cudaMemcpy(hf.data(), d_fate, 64, cudaMemcpyDeviceToHost));
      for (int i = 0; i < 8; ++i) hist->fate_count[i] += hf[i];
    }
    if (hist->total_steps) {
      DW_CUDA(c, cudaMemcpy(hs.data(), d_steps, 8, cudaMemcpyDeviceToHost));
      hist->total_steps[0] += hs[0];
    }
  }
  return DW_OK;
}
