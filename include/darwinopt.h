/* darwinopt.h -- C ABI of libdarwinopt.so: B200-native photon propagation through a triangle-mesh
 * detector, the hot path of "GPU-based optical simulation of the DARWIN detector" (arXiv 2203.14354).
 *
 * Citations: P:<n> = line n of the paper text; S<k>/G<k> = step / reading of DESIGN.md
 * section "Oracle and readings" (same numbering as SURVEY.md section 8(c)).
 *
 * What the calls are (section 1: "the core of the framework's photon propagation code is written in
 * CUDA C"; the problem statement: upload geometry and wavelength-tabulated optical properties, build the
 * acceleration structure, propagate a photon batch with a step limit, get per-channel hits and fates):
 *
 *   dw_create / dw_destroy            context on one CUDA device; owns every device copy it makes
 *   dw_set_materials                  n, L_abs, L_Rayleigh per material vs wavelength        (Table 2)
 *   dw_set_surfaces                   detect / diffuse / specular / transmit probabilities
 *   dw_set_films                      surfaces from a complex index and a film thickness    (Table 8)
 *   dw_set_geometry                   triangle mesh + per-triangle inner/outer material, surface, channel
 *   dw_build_bvh                      device LBVH build (one-off per geometry)
 *   dw_refit_bvh                      same triangles at new vertex positions, tree kept       (P:305-412 design sweeps)
 *   dw_first_hit                      nearest triangle along rays (S1) -- the parity entry of the query
 *   dw_render                         S1 for the rays of a pinhole camera: ids, depths, shaded image
 *   dw_propagate                      the Monte Carlo loop S1..S13 for a photon batch, device buffers
 *   dw_propagate_host                 same, host buffers (copies inside), for end-to-end timing
 *   dw_emit                           scintillation photons generated on the device          (Table 2)
 *   dw_tally / dw_tally_finish        counts per source and array, arrival-time histograms, loss table; LCE and t90 (Table 6)
 *   dw_emit_sources / dw_design_study many sources per launch; the whole emit -> propagate -> tally loop as one call
 *
 * Conventions
 *   - Units mm, ns, nm.  c = 299.792458 mm/ns.  All floating point is IEEE fp32.
 *   - Triangle normal n_g = normalize((v1-v0)x(v2-v0)) points from the INNER to the OUTER material.
 *   - Every function returns 0 (DW_OK) or a negative dw_status; nothing throws or aborts across the ABI.
 *     dw_last_error() gives a context-owned message valid until the next call on that context.
 *   - "host" / "device" is stated for every pointer.  The library never frees or keeps caller pointers
 *     after the call returns, except stream-ordered use: device buffers passed to an asynchronous call
 *     must stay alive until the stream has reached the end of that call's work.
 *   - Triangle ids in all outputs are the CALLER's numbering (the BVH leaf order is internal).
 *   - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream).
 *   - There is no CPU fallback: without a CUDA device dw_create fails with DW_E_CUDA.
 */
#ifndef DARWINOPT_H_
#define DARWINOPT_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct dw_ctx dw_ctx;

typedef enum dw_status {
  DW_OK = 0,
  DW_E_ARG = -1,    /* NULL / negative / inconsistent argument                                  */
  DW_E_STATE = -2,  /* call out of order (e.g. propagate before build_bvh, geometry before tables) */
  DW_E_CUDA = -3,   /* a CUDA runtime call failed; message in dw_last_error                     */
  DW_E_RANGE = -4   /* an index in the geometry is out of range, or a probability table is invalid */
} dw_status;

/* Photon fate = low 4 bits of the per-photon flags word; exactly one per photon (S10, S11, P9). */
enum {
  DW_FATE_DETECTED = 0,         /* hit a triangle with a surface, "detect" drawn        */
  DW_FATE_BULK_ABSORBED = 1,    /* absorbed in the medium (Table 2 L_abs)                        */
  DW_FATE_SURFACE_ABSORBED = 2, /* explicit surface, none of detect/reflect/transmit drawn       */
  DW_FATE_ESCAPED = 3,          /* ray left the world (G3)                                       */
  DW_FATE_TRUNCATED = 4,        /* max_steps reached                                             */
  DW_FATE_NAN_ABORT = 5,        /* non-finite state (must count 0)                               */
  DW_FATE_MASK = 0xF
};
/* History bits OR-ed into flags. */
enum {
  DW_H_RAYLEIGH = 0x10, DW_H_REFLECT_DIFFUSE = 0x20, DW_H_REFLECT_SPECULAR = 0x40,
  DW_H_SURFACE_TRANSMIT = 0x80, DW_H_FRESNEL_REFLECT = 0x100, DW_H_FRESNEL_REFRACT = 0x200,
  DW_H_TIR = 0x400,
  DW_H_MEDIUM_MISMATCH = 0x800, /* carried medium != medium seen from the hit triangle (ill-formed mesh) */
  DW_H_FILM = 0x1000            /* the last surface event was on a thin-film surface (with REFLECT_SPECULAR / SURFACE_TRANSMIT) */
};

int dw_create(int cuda_device, dw_ctx** out);
int dw_destroy(dw_ctx* ctx);
const char* dw_last_error(const dw_ctx* ctx); /* ctx may be NULL: message of the last failed dw_create */
int dw_version(void);

/* Materials on a uniform wavelength grid lambda0 + i*dlambda (i < n_lambda, n_lambda >= 1); values between
 * nodes are linearly interpolated and clamped at the ends (S3, G13).  Arrays are HOST pointers, row-major
 * [n_mat][n_lambda]; abs_len_mm / scat_len_mm = +inf switches the process off.  n_mat <= 255. */
int dw_set_materials(dw_ctx* ctx, int n_mat, int n_lambda, float lambda0, float dlambda,
                     const float* refr_index, const float* abs_len_mm, const float* scat_len_mm);

/* Explicit surfaces (reflectivity "explicitly specified (separately for diffuse and specular
 * components)", independent of the angle of incidence).  HOST pointers, [n_surf][n_lambda] each.  One uniform
 * number is compared with the cumulative sums in the order detect, reflect_diffuse, reflect_specular,
 * transmit; the remainder absorbs (S7).  DW_E_RANGE if an entry is < 0 or a sum exceeds 1 + 1e-6.
 * n_surf <= 254.  May be called again at any time (a design sweep changes reflectivities without a BVH
 * rebuild); the grid may differ from the materials' grid. */
int dw_set_surfaces(dw_ctx* ctx, int n_surf, int n_lambda, float lambda0, float dlambda,
                    const float* detect, const float* reflect_diffuse, const float* reflect_specular,
                    const float* transmit);

/* Thin-film surfaces.  PAPER.md line 175: surface reflectivity "calculated using Fresnel equations from the
 * specified complex index of refraction and surface thickness"; Table 8 (lines 356-357): silicon n = 0.81, k = 1.86.
 * For every surface s with film_on[s] != 0 the explicit probabilities are not used; instead a film of index n_film + i k_film
 * and thickness thickness_nm lies between the photon's medium (n1) and the material on the other side of the triangle (n3):
 * amplitudes by the single-film Airy summation per polarisation, R and T mixed by intensities as in S8; one uniform number
 * (u_fresnel) decides reflect (specular) / transmit (refracted into n3, the photon changes medium) / absorbed in the film, and an
 * absorbed photon is DETECTED with the surface's `detect` probability (u_surface), else SURFACE_ABSORBED.  History bit DW_H_FILM.
 * HOST pointers: film_on [n_surf], the three tables [n_surf][n_lambda] on the SAME grid as the last dw_set_surfaces (n_surf,
 * n_lambda, lambda0, dlambda must match it: DW_E_ARG otherwise; DW_E_STATE before dw_set_surfaces).  A later dw_set_surfaces with a
 * different shape drops the films.  k_film >= 0, thickness_nm >= 0, n_film > 0 (DW_E_RANGE).  film_on == NULL removes all films. */
int dw_set_films(dw_ctx* ctx, int n_surf, int n_lambda, float lambda0, float dlambda, const int32_t* film_on,
                 const float* n_film, const float* k_film, const float* thickness_nm);

/* Geometry: xyz [n_vert][3] fp32, idx [n_tri][3] int32, and per triangle the inner / outer material id,
 * the surface id (-1 = none: Fresnel between the two materials, S8) and the sensor channel (-1 = none).
 * pointers_are_device = 0: HOST pointers; 1: DEVICE pointers (read on the legacy default stream).
 * The data is copied; the caller keeps ownership.  Requires materials and surfaces to be set (ids are
 * validated against them): DW_E_STATE otherwise; DW_E_RANGE on an out-of-range index or id, a non-finite
 * vertex, or a zero-area triangle.  Invalidates a previous BVH. */
int dw_set_geometry(dw_ctx* ctx, int64_t n_vert, const float* xyz, int64_t n_tri, const int32_t* idx,
                    const int32_t* mat_inner, const int32_t* mat_outer, const int32_t* surface,
                    const int32_t* channel, int pointers_are_device);

typedef struct dw_build_params {
  int32_t max_leaf_tris; /* 1..8, triangles per BVH leaf; 0 = default (2) */
  int32_t ploc_radius;   /* 1..256, search radius of the clustering rounds in Morton order; 0 = default (16) */
  int32_t grid_res;      /* 8..128, cells per axis of the empty-space grid; 0 = default (64); -1 = no grid */
  int32_t split_div;     /* a triangle longer than (largest scene extent) / split_div gets several box references;
                          * 1..4096; 0 = default (32); -1 = never split.  Halved automatically while the references
                          * would exceed 2 n_tri + 65536. */
  int32_t reserved[4];
} dw_build_params;

typedef struct dw_build_stats {
  int64_t n_tri, n_nodes, node_bytes, tri_bytes;
  int32_t max_depth, n_leaves; /* max_depth: levels of the 4-wide traversal tree */
  float scene_lo[3], scene_hi[3];
  float build_ms; /* device time of the whole build */
  int32_t ploc_rounds;  /* clustering rounds executed */
  int32_t binary_depth; /* depth of the binary tree before the collapse into 4-wide nodes */
  int32_t grid_res;        /* cells per axis of the empty-space grid actually built (0 = none) */
  int32_t grid_free_cells; /* cells that got a triangle-free box */
  int32_t n_refs;          /* box references the tree is built over (>= n_tri); tri_bytes = 48 * n_refs */
  int32_t split_div;       /* divisor actually used (0 = nothing was split) */
} dw_build_stats;

/* Device LBVH build: triangle boxes -> scene bounds -> 63-bit Morton codes of the centroids -> radix sort ->
 * binary radix tree -> bottom-up refit -> traversal nodes + triangles permuted to leaf order.
 * params NULL = defaults; stats may be NULL.  Synchronises the stream before returning (one-off call). */
int dw_build_bvh(dw_ctx* ctx, const dw_build_params* params, dw_build_stats* stats, void* cuda_stream);

typedef struct dw_refit_stats {
  float refit_ms;          /* device time of the whole refit (upload of the vertices included) */
  int32_t n_levels;        /* levels of the 4-wide tree whose boxes were recomputed */
  int32_t n_loose_tris;    /* split triangles whose number of pieces changed (split more coarsely, or pieces shared by references) */
  int32_t grid_free_cells; /* cells of the rebuilt empty-space grid that got a triangle-free box (0 without a grid) */
  float scene_lo[3], scene_hi[3];
  float area_ratio;        /* sum of the half-areas of all child boxes of the tree, relative to the same sum when the tree was built:
                            * the expected box tests per ray grow with it; well above 1 means a rebuild pays */
} dw_refit_stats;

/* Geometry variants without a rebuild (the paper's design sweeps move or reshape components of one detector,
 * P:305-412): new vertex positions xyz [n_vert][3] for the SAME triangles (indices, materials, surfaces and channels as set by
 * dw_set_geometry; n_vert must match).  The tree keeps its shape; triangle records, reference boxes (long triangles are clipped
 * again; a changed piece count is fitted to the references the tree has), the boxes of all 4-wide nodes bottom-up, the length
 * tolerance and the empty-space grid are recomputed.  The tree only decides HOW the nearest hit is found: every query gives the
 * result a fresh dw_build_bvh on the moved geometry gives, bit for bit; large motions cost speed, not correctness.
 * pointers_are_device as in dw_set_geometry.  DW_E_STATE before dw_build_bvh; DW_E_ARG on a size mismatch; DW_E_RANGE on a
 * non-finite vertex or a zero-area triangle (the context then has no BVH and no valid geometry: set it again).  Synchronises. */
int dw_refit_bvh(dw_ctx* ctx, int64_t n_vert, const float* xyz, int pointers_are_device, dw_refit_stats* stats, void* cuda_stream);

/* First hit (S1): for ray i the triangle with the smallest d > 0 along o + d*dir, ignoring triangle
 * exclude_tri[i] (caller id; pointer may be NULL); exact ties -> lowest caller id.  DEVICE pointers, length n.
 * Miss: tri_out = -1, dist_out = +inf.  Asynchronous on the stream. */
int dw_first_hit(dw_ctx* ctx, int64_t n, const float* ox, const float* oy, const float* oz,
                 const float* dx, const float* dy, const float* dz, const int32_t* exclude_tri,
                 int32_t* tri_out, float* dist_out, void* cuda_stream);

/* Ray cast of the mesh into device buffers (the "Chroma rendering" insert of Fig. 1, without
 * a display): a pinhole camera at `eye` looking along `forward`, image `width` x `height` pixels, vertical field of view fov_y_deg.
 * With f = unit(forward), r = unit(f x up), u = r x f, t = tan(fov_y / 2), the ray of pixel (i, j) -- i to the right, j downwards,
 * stored at [j * width + i] -- has direction unit(f + x t (width / height) r + y t u), x = 2 (i + 0.5) / width - 1,
 * y = 1 - 2 (j + 0.5) / height, and is answered by the first-hit query S1 (no excluded triangle). */
typedef struct dw_camera {
  float eye[3], forward[3], up[3];
  float fov_y_deg;
  int32_t width, height;
} dw_camera;
/* Outputs are DEVICE pointers of width * height elements, any may be NULL: tri_out = caller id of the nearest triangle or -1,
 * depth_out = its distance or +inf, shade_out = round(255 |n . d|) with n the unit normal of that triangle, 0 on a miss.
 * DW_E_STATE before dw_build_bvh; DW_E_ARG for a bad size (1..32768), field of view, or an up vector parallel to forward.
 * Asynchronous on the stream. */
int dw_render(dw_ctx* ctx, const dw_camera* camera, int32_t* tri_out, float* depth_out, uint8_t* shade_out, void* cuda_stream);

/* Photon batch, structure of arrays, each of length n (52 B per photon).  Directions and polarisations are
 * unit vectors with pol . dir = 0.  photon_id_base + i is photon i's identity in the counter-based random
 * number generator (Philox4x32-10, key = seed, counter = (id lo, id hi, step, block)), so that splitting or
 * permuting a batch does not change any photon's result. */
typedef struct dw_photons {
  int64_t n;
  uint64_t photon_id_base;
  const float *px, *py, *pz;   /* position, mm     */
  const float *kx, *ky, *kz;   /* direction        */
  const float *ex, *ey, *ez;   /* polarisation     */
  const float* wavelength;     /* nm               */
  const float* t0;             /* start time, ns   */
} dw_photons;

/* Per-photon results, each of length n; any pointer may be NULL (not written). */
typedef struct dw_results {
  uint32_t* flags;    /* fate | history bits                                  */
  int32_t* channel;   /* sensor channel if DETECTED else -1                   */
  float* t;           /* time at the end of the track, ns                     */
  uint32_t* steps;    /* loop iterations executed, including the terminating one */
  int32_t* last_tri;  /* caller id of the last surface touched, -1 if none / after a scatter */
  float *x, *y, *z;   /* final position                                       */
  float *kx, *ky, *kz;/* final direction   (diagnostic)                       */
  float *ex, *ey, *ez;/* final polarisation (diagnostic)                      */
} dw_results;

/* Reductions (S13).  All ACCUMULATED into: the caller zeroes them, so that the batches of a sweep add up.
 * Any pointer may be NULL. */
typedef struct dw_hists {
  int64_t n_chan;          /* length of chan_count; detected photons with channel outside [0,n_chan) are not counted */
  uint64_t* chan_count;    /* [n_chan] photons DETECTED per channel                                 */
  int64_t n_bins;          /* length of time_hist                                                   */
  float t_min, dt;         /* bin = floor((t - t_min)/dt) clamped to [0, n_bins-1]                  */
  uint32_t* time_hist;     /* [n_bins] arrival times of detected photons                            */
  uint64_t* fate_count;    /* [8] photons per fate code                                             */
  uint64_t* total_steps;   /* [1] photon-steps executed                                             */
} dw_hists;

typedef struct dw_propagate_params {
  uint32_t flags;          /* DW_PROP_* */
  int32_t block_threads;   /* 0 = default */
  int32_t blocks_per_sm;   /* 0 = default */
  int32_t th_phys;         /* pool scheduler (default): idle lanes of a warp that trigger a refetch of queued rays or the
                            * physics phase; legacy scheduler: lanes waiting for physics that trigger it; 0 = default */
  int32_t th_leaf;         /* run the triangle phase once this many lanes of a warp wait for it; 0 = default */
  int32_t reserved[3];
} dw_propagate_params;
enum {
  /* Follow the oracle's loop literally (S1..S4 in its order): every query is unbounded, the medium is read from the side of the hit
   * triangle (S2), and the bulk lengths compete with the hit distance afterwards.  One concession to fp32: right after a surface
   * event a triangle whose near side is not the medium the photon was just sent into is not a candidate (the hit point can lie
   * 1e-4 mm behind a neighbouring facet; in fp64 that hit does not exist).  A hit from the bulk on a side that contradicts the
   * carried medium is accepted and reported with DW_H_MEDIUM_MISMATCH: the test for an ill-formed mesh.
   * Default (flag clear): the medium is carried in the photon state after the first query and the sampled bulk distance bounds
   * the ray; equal in distribution in a closed world. */
  DW_PROP_UNBOUNDED_QUERY = 1u,
  /* Diagnostic: run the first-generation kernel (photon state in registers, one photon per lane, physics and
   * traversal phases chosen per warp) instead of the pool scheduler.  Same results photon by photon. */
  DW_PROP_LEGACY_SCHEDULER = 2u,
  /* Diagnostic: never answer a bounded query from the empty-space grid (every query is traversed).  Same results. */
  DW_PROP_NO_EMPTY_SKIP = 4u
};

/* The propagation loop S1..S13 for every photon of the batch, at most max_steps iterations each.
 * DEVICE pointers throughout.  Asynchronous on the stream; no host synchronisation inside.
 * params / out / hist may be NULL. */
int dw_propagate(dw_ctx* ctx, const dw_photons* in, uint64_t seed, int32_t max_steps,
                 const dw_results* out, const dw_hists* hist, const dw_propagate_params* params,
                 void* cuda_stream);

/* Same computation with HOST pointers in `in`, `out` and `hist` (pinned memory recommended): the call copies
 * the batch to the device in chunks overlapped with propagation, copies the requested results back and ADDS
 * the reductions into the host arrays.  Synchronous: returns when the host buffers are complete.
 * Chunks: 1 Mi photons first, then three times larger each time up to 6 Mi (environment: DW_HOST_FIRST, DW_HOST_CHUNK, in photons;
 * DW_HOST_SLOTS = 2..4 staging buffers); the context keeps 2 x 100 B x chunk of device staging memory (1.26 GB at the default). */
int dw_propagate_host(dw_ctx* ctx, const dw_photons* in, uint64_t seed, int32_t max_steps,
                      const dw_results* out, const dw_hists* hist, const dw_propagate_params* params);


/* Emission of scintillation photons on the device.
 * "The emission spectrum is modeled as a Gaussian with a mean of 174.8 nm and a full width at half maximum of
 * 10.2 nm.  The scintillation time profile is modeled by a two-component exponential decay function"; Table 2 (lines 155-160):
 * tau_1 = 3.5 ns, tau_3 = 24 ns, singlet fraction 0.66 (nuclear recoils) / 0.22 (electronic recoils); line 191: photons are
 * generated isotropically and uniformly in the active region.
 * Photon photon_id_base + i takes Philox blocks 0..2 of the reserved step 0xFFFFFFFF (key = seed), so the result depends on
 * (seed, photon id) only and any split of a batch gives the same photons:
 *   position   shape 0: centre; 1: uniform in the cylinder of `radius` about the z axis through centre, z in [z0, z1];
 *              2: uniform in the ball of `radius` about centre
 *   direction  isotropic;  polarisation  normalize(k x r) for an independent isotropic r (random transverse)
 *   wavelength lambda_mean + lambda_sigma * N(0,1) (Box-Muller; sigma = FWHM / (2 sqrt(2 ln 2)); not truncated)
 *   time       t_start - tau ln u with tau = tau1 with probability f_singlet, else tau3 */
typedef struct dw_source {
  int32_t shape;                 /* DW_SOURCE_* */
  float centre[3];               /* mm */
  float radius, z0, z1;          /* mm; z0 <= z1 (cylinder only) */
  float lambda_mean, lambda_sigma; /* nm; sigma >= 0 */
  float t_start, tau1, tau3;     /* ns; tau >= 0 */
  float f_singlet;               /* in [0, 1] */
  int32_t reserved[3];
} dw_source;
enum { DW_SOURCE_POINT = 0, DW_SOURCE_CYLINDER = 1, DW_SOURCE_BALL = 2 };

/* Writes out->n photons into the eleven DEVICE arrays of `out` (they are written although the struct declares them const:
 * the same struct then goes to dw_propagate).  Asynchronous on the stream.  DW_E_ARG for a bad source or a null array. */
int dw_emit(dw_ctx* ctx, const dw_source* source, uint64_t seed, const dw_photons* out, void* cuda_stream);


/* Design-study reductions over the per-photon results of dw_propagate.
 * "LCE is defined here as the number of photons hitting the photosensitive area divided by the total number of
 * generated photons", reported per source position and separately for the top and bottom arrays (lines 249-253: ~2500 point sources
 * on a Z x R^2 grid); line 211: t90, "the time to collect 90% of detected photons"; lines 267-271 and Table 6: where the photons that
 * are not detected get absorbed, by component.  Photon i belongs to source i / photons_per_source (the last source may be short).
 *   detected[s][g]            photons of source s DETECTED on a channel c with channel_group[c] == g      (LCE = detected / generated)
 *   time_hist[s][b]           arrival times of the DETECTED photons of source s, b = floor((t - t_min) / dt) clamped to [0, n_bins)
 *   fate_by_source[s][f]      photons of source s with fate f (8 columns; bulk absorption is column DW_FATE_BULK_ABSORBED)
 *   absorbed_by_component[k]  SURFACE_ABSORBED photons whose last triangle t has tri_component[t] == k
 * Everything is ACCUMULATED (the caller zeroes) and integer, so sweeps add up and the result is bit-reproducible.  All pointers are
 * DEVICE pointers; flags is required, channel / t / last_tri only for the tables that use them; any output may be NULL.  Channels or
 * triangles outside [0, n_chan) / [0, n_tri_map), and groups or components outside their range, are not counted.  Asynchronous. */
typedef struct dw_tally_tables {
  const int32_t* channel_group;  int64_t n_chan;     int32_t n_groups;      /* [n_chan]     */
  const int32_t* tri_component;  int64_t n_tri_map;  int32_t n_components;  /* [n_tri_map], indexed by the caller's triangle id */
  uint64_t* detected;            /* [n_sources][n_groups] */
  uint32_t* time_hist;  int64_t n_bins;  float t_min, dt;                    /* [n_sources][n_bins] */
  uint64_t* fate_by_source;      /* [n_sources][8] */
  uint64_t* absorbed_by_component; /* [n_components] */
} dw_tally_tables;
int dw_tally(dw_ctx* ctx, const dw_results* results, int64_t n, int64_t photons_per_source, const dw_tally_tables* tables,
             void* cuda_stream);

/* The two products the paper derives from those tables, computed on the device ("on-device LCE(Z,R^2) and t90
 * maps").  PAPER.md line 189: "LCE is defined here as the number of photons hitting the photosensitive area divided by the total
 * number of generated photons"; line 211: t90 is "the time to collect 90% of detected photons".
 *   lce_out[s][g] = detected[s][g] / generated[s],  generated[s] = sum over the 8 columns of fate_by_source[s]   (NaN if 0 generated)
 *   t90_out[s]    = the time by which the fraction `quantile` (0.9 for t90) of the photons counted in time_hist[s] has arrived.
 *                   Reading T-t90 (the paper gives a definition, no estimator): with N = sum of the row and c(b) the count of bins
 *                   0..b, take the first bin b with c(b) >= quantile N and place the crossing linearly inside it:
 *                   t = t_min + dt (b + (quantile N - c(b-1)) / time_hist[s][b]).  NaN if the row is empty.  Underflow and overflow
 *                   photons sit in the first and last bin (dw_tally clamps), so choose the range to hold the quantile.
 * Sums and the division are done in double precision and rounded to fp32 once.  tables: the struct given to dw_tally (its detected,
 * fate_by_source, time_hist, n_groups, n_bins, t_min, dt are read; nothing is modified).  lce_out [n_sources][n_groups] needs detected
 * and fate_by_source, t90_out [n_sources] needs time_hist; either output may be NULL.  DEVICE pointers.  0 < quantile <= 1.
 * Asynchronous on the stream. */
int dw_tally_finish(dw_ctx* ctx, const dw_tally_tables* tables, int64_t n_sources, float quantile, float* lce_out, float* t90_out,
                    void* cuda_stream);

/* Many sources per launch ("close to 2500" point sources on a Z x R^2 grid, 1e6 photons
 * each).  dw_emit for photon i of source i / photons_per_source, in ONE launch: out->n photons (at most n_sources *
 * photons_per_source; the last source may be short), photon identity out->photon_id_base + i exactly as in dw_emit, so the photons are
 * bit-identical to n_sources separate dw_emit calls with id bases out->photon_id_base + s * photons_per_source.
 * sources: HOST pointer [n_sources] (copied to the device on the stream before the launch); out: DEVICE arrays.  Asynchronous,
 * except that a pageable host array is read before the call returns. */
int dw_emit_sources(dw_ctx* ctx, const dw_source* sources, int64_t n_sources, int64_t photons_per_source, uint64_t seed,
                    const dw_photons* out, void* cuda_stream);

/* The design-study loop of PAPER.md sections 4.1-4.2 (lines 189, 211, 249-253, 267-271) as one call: for sources_per_batch sources
 * at a time dw_emit_sources -> dw_propagate -> dw_tally into `tables` (rows = sources, ACCUMULATED: the caller zeroes), then
 * dw_tally_finish.  Photon ids are s * photons_per_source + i for photon i of source s, so no result depends on sources_per_batch.
 * sources: HOST [n_sources]; tables and lce_out / t90_out (may be NULL): DEVICE.  sources_per_batch <= 0: as many as fit 2^25 photons.
 * The call allocates and frees its photon and result buffers on the stream (60 B per photon of a batch).  Asynchronous like
 * dw_emit_sources. */
int dw_design_study(dw_ctx* ctx, const dw_source* sources, int64_t n_sources, int64_t photons_per_source, uint64_t seed,
                    int32_t max_steps, const dw_tally_tables* tables, int64_t sources_per_batch, float quantile, float* lce_out,
                    float* t90_out, void* cuda_stream);

/* dw_design_study for callers that may not allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc): the same
 * loop and the same results (photon ids are s * photons_per_source + i, so the batching does not show), but the source table, the
 * photon and result buffers of a batch and the queue head of the propagation launches lie in ONE file-scope device array of
 * DW_STATIC_SCRATCH_BYTES that every GPU on which the library's module is loaded holds until the process exits.  The call makes no
 * cudaMalloc / cudaFree / cudaMallocAsync and creates no stream or event; it issues one cudaMemcpyAsync (the sources), 8-byte
 * cudaMemsetAsync's and kernel launches on the stream.  Limits, DW_E_RANGE with a message beyond them:
 *   n_sources <= DW_STATIC_MAX_SOURCES,  photons_per_source <= DW_STATIC_MAX_PHOTONS (a batch is as many whole sources as fit that).
 * sources: HOST [n_sources]; tables (ACCUMULATED: the caller zeroes) and lce_out / t90_out (may be NULL): DEVICE, the caller's.
 * The array is shared by ALL contexts and calls on a device and keeps the last call's contents: the call zeroes the queue head
 * before every launch and overwrites what it reads, but two calls that overlap on the GPU (different streams, or two contexts on
 * one device) race on it -- keep them on one stream or order them with events.  The first call on a device looks the array up
 * (cudaGetSymbolAddress with that device current, which loads the module); make one call before a capture starts.  Asynchronous
 * like dw_emit_sources. */
#define DW_STATIC_MAX_SOURCES 4096
#define DW_STATIC_MAX_PHOTONS 262144
#define DW_STATIC_SCRATCH_BYTES (256 + 64 * DW_STATIC_MAX_SOURCES + 60 * DW_STATIC_MAX_PHOTONS)   /* 15.25 MiB */
int dw_design_study_static(dw_ctx* ctx, const dw_source* sources, int64_t n_sources, int64_t photons_per_source, uint64_t seed,
                           int32_t max_steps, const dw_tally_tables* tables, float quantile, float* lce_out, float* t90_out,
                           void* cuda_stream);


/* Measured denominators for the roofline (SURVEY.md 8(d) "Peaks": the driver's peaks file holds HBM and
 * tensor numbers only).  Runs four short register-only / L2-resident kernels on the default stream and waits for them:
 *   out[0] FP32 FMA lane-instructions / s        out[1] integer ALU (LOP3) lane-instructions / s
 *   out[2] lane-instructions / s of an even FMA + ALU mix (what the propagation kernel issues)
 *   out[3] bytes / s read from a 32 MiB buffer that stays in L2
 * About 0.1 s.  Not part of the hot path. */
int dw_probe_peaks(dw_ctx* ctx, double out[4]);

/* Diagnostics for the roofline line ("n_node and n_tri are measured by an instrumented build of the kernel"): runs the
 * counting instantiation of the default propagation kernel once over `in` (DEVICE arrays; no per-photon outputs, no histograms) on the
 * legacy default stream, waits, and writes DW_N_COUNTERS values to the HOST array counters_out:
 *   [0] box-node visits  [1] ray-triangle tests  [2] queries traversed  [3] queries answered by the empty-space grid
 *   [4] physics phases  [5] finished queries evaluated in them  [6] lanes that ran an iteration of the Rayleigh loop
 *   [7] queries set up  [8] photons loaded  [9,10] iterations and active lanes of the box-node phase of the traversal loop
 *   [11,12] the same of its triangle phase  [13] fetches of queued queries  [14] unused  [15] physics phases that ran a Rayleigh iteration
 *   [16,17] first (unbounded) queries of photons and their node visits  [18,19,20] queries that start on a surface, their node
 *   visits, those that hit something  [21,22,23] the same for queries that start in the bulk
 * Several times slower than dw_propagate (shared-memory atomics per event); never part of a timed region. */
enum { DW_N_COUNTERS = 24 };
int dw_propagate_counters(dw_ctx* ctx, const dw_photons* in, uint64_t seed, int32_t max_steps, const dw_propagate_params* params,
                          uint64_t* counters_out);

/* Diagnostics / tests: raw Philox4x32-10 blocks and the uniforms the kernel derives from them, computed on the
 * device.  out_raw [n][4] uint32, out_u [n][4] float (either may be NULL), DEVICE pointers; entry i uses
 * photon id photon_id_base + i, the given step and block. */
int dw_debug_philox(dw_ctx* ctx, uint64_t seed, uint64_t photon_id_base, uint32_t step, uint32_t block,
                    int64_t n, uint32_t* out_raw, float* out_u, void* cuda_stream);

/* Last kernel launch configuration used by dw_propagate (grid, block, dynamic smem bytes, kernels launched). */
int dw_last_launch(const dw_ctx* ctx, int32_t* grid, int32_t* block, int32_t* smem_bytes, int64_t* n_launches);

#ifdef __cplusplus
}
#endif
#endif /* DARWINOPT_H_ */
