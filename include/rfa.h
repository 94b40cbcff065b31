/*
 * rfa.h -- C ABI of librfa.so: explicit finite-difference stepping of the simplified bioheat
 * equation of arXiv 1907.05709 (Kath, Handels, Mastmeyer) on a labelled voxel volume, on one
 * NVIDIA B200 (sm_100a).  Plain pointers and sizes only; no C++ or torch types cross this boundary.
 *
 * What one time step computes (citations: line numbers of the paper text, PAPER.md):
 *   for every voxel v = (i,j,k) of every scenario
 *     held voxel (vessel / fixed label / Dirichlet needle voxel):   T^{n+1} = T^n       Eq. 13 :122-125, Alg. 1 :313
 *     otherwise  T^{n+1} = T^n + dt/(rho c_p) * [ K * ( d2x + d2y + d2z )               Eq. 12 :117
 *                                  + w_b c_b (T_a - T^n) + Q_m (+ Q in POWER voxels) ]   Eq. 9  :102
 *       d2x = (T_{i-1} - 2 T_i + T_{i+1}) / dx^2  etc.                                   Eq. 11 :112
 *       rho, c_p, K, w_b c_b, Q_m looked up from the voxel's label ("voxel-wise", :120)
 *       outer grid faces: zero flux, the missing neighbour is the voxel itself (R-7)
 *     necrosis[v] |= (T^{n+1} >= 60 C), sticky                                           :37, R-11/R-12
 *   two temperature buffers are ping-ponged (Alg. 2 :321-337).
 *
 * Layout: every volume is x fastest, idx = i + nx*(j + ny*k); batched volumes are scenario-major.
 * Arithmetic: fp32 on the device, stored as theta = T - t_blood (exact shift of the affine PDE,
 * DESIGN.md section 5); per-label coefficients are derived in fp64 on the host and rounded once.
 *
 * Memory: "host" pointers are ordinary host memory.  Pointers documented "host or device" may be
 * either (the library asks the CUDA runtime).  Host inputs are copied during the call; device inputs are
 * read asynchronously on the simulation's stream (stated per call); the caller keeps ownership of all its
 * buffers.  A simulation lives on the CUDA device that is current at rfa_create: every later call switches
 * to that device for its own work and restores the caller's current device before it returns.  Device state lives in the caller's workspace
 * (see rfa_workspace_bytes) or, if none is given, in memory the library allocates and frees.
 *
 * Errors: every int-returning call returns RFA_OK (0) or a negative code; no exception crosses the
 * ABI and a failed rfa_create leaves nothing allocated.  rfa_last_error() gives the message of the
 * calling thread's last failure.  rfa_step is asynchronous on the simulation's stream; the rfa_get_*,
 * rfa_necrotic_voxels and rfa_synchronize calls wait for it.
 */
#ifndef RFA_H
#define RFA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rfa_sim rfa_sim; /* opaque */

/* One row per label id, SI units (constants of PAPER.md:104). 28 bytes, no padding. */
typedef struct rfa_tissue {
    float k;        /* W/(m K)    thermal conductivity K                                    */
    float rho;      /* kg/m^3     tissue density                                            */
    float cp;       /* J/(kg K)   tissue heat capacity c_p                                  */
    float wb_cb;    /* W/(m^3 K)  perfusion sink coefficient  w_b * c_b  of Eq. 9           */
    float q_m;      /* W/m^3      metabolic heat Q_m                                        */
    float t_init;   /* deg C      initial temperature of this label (Fig. 5)  */
    uint32_t flags; /* RFA_TISSUE_HELD: never updated, stays at its temperature (Eq. 13)    */
} rfa_tissue;

enum { RFA_TISSUE_HELD = 1 };
enum { RFA_MAX_TISSUES = 16 };   /* label ids 0..15 (4 bits of the packed state byte) */

/* needle source modes (PAPER.md:145 held tip; BASELINE.json config 3 constant power, R-17) */
enum { RFA_SRC_OFF = 0, RFA_SRC_DIRICHLET = 1 /* value = deg C */, RFA_SRC_POWER = 2 /* value = W/m^3 */ };

enum {
    RFA_OK = 0,
    RFA_E_INVALID = -1,   /* null pointer, non-positive dims/spacing/dt, label >= n_tissue, > 16 tissues,
                             scenario out of range, bad mode, workspace too small, non-finite constants */
    RFA_E_UNSTABLE = -2,  /* dt violates the monotone bound dt*(2 alpha sum 1/h^2 + w_b c_b/(rho c_p)) <= 1
                             for some non-held label (R-18)                                    */
    RFA_E_CUDA = -3,      /* a CUDA runtime call or kernel launch failed (also: no device)              */
    RFA_E_NOMEM = -4      /* host or device allocation failed                                          */
};

/* conduction term (rfa_set_conduction) */
enum {
    RFA_COND_EQ12 = 0,        /* Eq. 12 as printed: the voxel's own K times the 7-point Laplacian; default */
    RFA_COND_FACE = 1         /* div(K grad T) of Eq. 9, conservative: flux through a face =
                                 Kf (T_n - T_c)/h with the harmonic mean Kf = 2 K_c K_n/(K_c + K_n) of the two
                                 voxels' K; identical to Eq. 12 inside a tissue, differs only at interfaces
                                 (R-28).  Conserves sum rho c_p T.            */
};

/* kernel variants for rfa_configure (all produce bit-identical fields) */
enum {
    RFA_KERNEL_AUTO = 0,      /* temporally blocked kernel where the grid allows it, else the plain one */
    RFA_KERNEL_PLAIN = 1,     /* one thread per voxel, one step per launch, global loads only          */
    RFA_KERNEL_BLOCKED = 2,   /* 2.5D z-sweep with register queues, fused_steps time steps per launch   */
    RFA_KERNEL_STREAM = 3     /* one time step per launch (the frame loop of Alg. 2), 128 x 32 tiles with
                                 halos staged in shared memory by the Tensor Memory Accelerator; needs nx % 16 == 0 and
                                 RFA_COND_EQ12.  RFA_KERNEL_AUTO uses it for every single-step launch where it applies
                                 (fused_steps = 1, and the remainder launch of n % fused_steps = 1)               */
};

/* Bytes of device workspace rfa_create needs for these dims (nx,ny,nz) and batch; 0 on bad input. */
size_t rfa_workspace_bytes(const int dims[3], int batch);

/* Monotone stability number  max over non-held labels of  dt*(2 K/(rho c_p) (1/dx^2+1/dy^2+1/dz^2)
 * + w_b c_b/(rho c_p));  rfa_create rejects values > 1 (R-18).  Host only, no GPU needed.
 * Returns a negative value on invalid input. */
double rfa_stability_number(const float spacing_mm[3], const rfa_tissue *table, int n_tissue, float dt_s);

/* Create a simulation of `batch` independent scenarios that share one label volume.
 *   dims        nx, ny, nz (> 0; ny, nz <= 65535)
 *   spacing_mm  voxel spacing in millimetres, converted to metres internally
 *   labels      host, nx*ny*nz bytes, label ids < n_tissue
 *   table       host, n_tissue rows (<= RFA_MAX_TISSUES)
 *   t_blood_c   T_a of Eq. 9 (deg C); dt_s the time step (s)
 *   workspace   device memory of >= rfa_workspace_bytes(dims,batch) bytes, 256-byte aligned, owned by
 *               the caller and kept alive until rfa_destroy; or NULL (the library allocates)
 *   cuda_stream a cudaStream_t (NULL = default stream); all work of this simulation runs on it
 * Initial state: T = t_init of the label, no needle, necrosis = (T >= 60). */
int rfa_create(rfa_sim **out, const int dims[3], const float spacing_mm[3], const uint8_t *labels,
               const rfa_tissue *table, int n_tissue, float t_blood_c, float dt_s, int batch,
               void *workspace, size_t workspace_bytes, void *cuda_stream);

/* Place (or move, or with RFA_SRC_OFF remove) the needle of one scenario.
 *   tip_mm, axis  metadata (the mask is authoritative), validated when given: tip_mm must lie inside the grid
 *                 [0, n*spacing] mm per axis and |axis| must be 1 +- 1e-3, else RFA_E_INVALID; either may be NULL
 *   mask          host or device, nx*ny*nz bytes, nonzero = electrode voxel; ignored for RFA_SRC_OFF.
 *                 A host mask is copied before the call returns.  A DEVICE mask is read asynchronously on the
 *                 simulation's stream: keep it valid and unchanged until rfa_synchronize (or a stream event).
 *   DIRICHLET: mask voxels are set to `value` deg C and held, overriding the label (R-15)
 *   POWER:     mask voxels get +value W/m^3 in the bracket of Eq. 12; a held label stays held (R-17)
 * Voxels of a previous needle are released: they keep their temperature and follow their label (R-16). */
int rfa_set_needle(rfa_sim *s, int scenario, const float tip_mm[3], const float axis[3],
                   const uint8_t *mask, int mode, float value);

/* Overwrite the temperature image of one scenario (deg C, host or device, nx*ny*nz floats);
 * necrosis |= (T >= 60).  Held voxels keep whatever is written here.  A host image is copied before the call
 * returns; a DEVICE image is read asynchronously on the simulation's stream (keep it valid until rfa_synchronize
 * or a stream event). */
int rfa_set_temperature(rfa_sim *s, int scenario, const float *t_c);

/* Advance every scenario by n time steps (n >= 0).  Asynchronous. */
int rfa_step(rfa_sim *s, int n);

/* Current temperature image (deg C) / necrosis mask (0 or 1) of one scenario into `out`
 * (host or device, nx*ny*nz elements). */
int rfa_get_temperature(rfa_sim *s, int scenario, float *out);
int rfa_get_necrosis(rfa_sim *s, int scenario, uint8_t *out);

/* Necrotic voxel counts of one scenario: all voxels of the mask, and those that are neither needle
 * voxels nor held labels (the reported necrotic volume, R-13).  Either pointer may be NULL. */
int rfa_necrotic_voxels(rfa_sim *s, int scenario, int64_t *all_voxels, int64_t *tissue_voxels);

/* Choose the kernel variant and, for the blocked kernel, the number of fused time steps (1..4; 0 = default).
 * RFA_KERNEL_STREAM takes fused_steps 0 or 1 and is rejected (RFA_E_INVALID) where it does not apply. */
int rfa_configure(rfa_sim *s, int kernel, int fused_steps);

/* Choose the conduction term for all scenarios (RFA_COND_*).  RFA_COND_FACE re-checks the monotone bound with
 * the largest face conductivity a voxel of each label can see (2 K K_max/(K + K_max)) and returns
 * RFA_E_UNSTABLE, leaving the mode unchanged, if dt violates it. */
int rfa_set_conduction(rfa_sim *s, int mode);

/* Introspection: fused steps in use, kernel in use, number of kernel launches issued so far by this simulation. */
int rfa_query(rfa_sim *s, int *kernel, int *fused_steps, int64_t *kernel_launches);

/* The variant rfa_step launches for this simulation:
 * out = { fused_steps, tile_bx, tile_by, ctas_launched, held_copy, conduction, staging (RFA_STAGING_CP_ASYNC / _TMA),
 *         residual_prefetch (0 / 1: what the next launch takes) }.  held_copy = 1: the kernel variant in
 * which warps whose voxels are all held copy their rows instead of evaluating the bracket (Alg. 1's else-branch,
 * PAPER.md:313; bit-identical), chosen at rfa_create when at least 1/8 of the volume carries a held label
 * (rfa_configure_held_copy overrides, for A/B measurements).  Zeros for the plain kernel. */
int rfa_query_variant(rfa_sim *s, int out[8]);

/* Force the held-copy kernel variant on or off, or hand the choice back to the library (what rfa_create decided
 * from the share of held labels).  All settings give bit-identical fields; the library reads no environment variable. */
enum { RFA_HELD_COPY_AUTO = -1, RFA_HELD_COPY_OFF = 0, RFA_HELD_COPY_ON = 1 };
int rfa_configure_held_copy(rfa_sim *s, int mode);

/* How the temporally blocked kernel brings the planes of the input image and the state bytes into shared memory (load step
 * of Alg. 1): per-thread cp.async, or one bulk tensor copy (Tensor Memory Accelerator) per tile plane issued by
 * a single thread.  The TMA variant exists for 2 and 3 fused steps in RFA_COND_EQ12 mode on grids with nx % 16 == 0 and ny
 * even; AUTO (the default) takes it where it measured faster (the 128 x 16 tile).  All settings give bit-identical fields.  Returns RFA_E_INVALID,
 * leaving the setting unchanged, when RFA_STAGING_TMA is asked for a grid that has no such variant.  The setting is kept across
 * rfa_set_conduction: while RFA_COND_FACE is active it has no effect (that mode has cp.async variants only; rfa_query_variant
 * shows the staging that really runs). */
enum { RFA_STAGING_AUTO = -1, RFA_STAGING_CP_ASYNC = 0, RFA_STAGING_TMA = 1 };
int rfa_configure_staging(rfa_sim *s, int mode);

/* Residual-prefetch variant of the blocked kernel (2 and 3 fused steps): the fp16 residual rows (compensated accumulation,
 * DESIGN.md section 5) of planes with |T - T_a| >= 1 C are fetched one plane ahead instead of where they are used.  It pays
 * where a few percent or more of the volume is that warm and costs ~3 % where next to nothing is, so in AUTO (the default) the
 * library switches it on and off from the share of such planes that the kernels count as they run (no synchronisation:
 * the count is copied to pinned memory asynchronously and looked at when it has arrived; in AUTO mode rfa_step stops
 * running more than ~64 launches ahead of the device, which always has 32 launches queued).  All settings give bit-identical
 * fields.  rfa_query_hot_fraction returns the last share seen and the variant in use (either pointer may be NULL). */
enum { RFA_RES_PREFETCH_AUTO = -1, RFA_RES_PREFETCH_OFF = 0, RFA_RES_PREFETCH_ON = 1 };
int rfa_configure_residual_prefetch(rfa_sim *s, int mode);
int rfa_query_hot_fraction(rfa_sim *s, double *fraction, int *prefetch_on);

/* Force the tile shape of the blocked kernel: 0 = 64 x 32 voxels (16 x 16 threads), 1 = 128 x 16 (32 x 8 threads), -1 = the
 * planner's choice (the default).  For A/B measurements; all shapes give bit-identical fields.  RFA_E_INVALID, leaving the
 * setting unchanged, if the shape cannot run the configured number of fused steps on this grid in the active conduction mode
 * (checked for every kernel setting except RFA_KERNEL_PLAIN, which has no tiles). */
int rfa_configure_tile(rfa_sim *s, int shape);

/* Host-only view of the blocked kernel's launch plan for a grid (no GPU needed; used by the unit tests
 * and the bench report).  resident_ctas = CTAs that can be co-resident (SM count x occupancy).
 * out = { ok, tiles_x, tiles_y, z_chunks, planes_per_chunk, work_items, ctas_launched, tile_bx, tile_by }. */
int rfa_plan_query(const int dims[3], int batch, int fused_steps, int resident_ctas, int staging, int out[9]);

/* ---- probe time series and frame hand-off ---------------------------------
 * The paper reads temperatures at probe points 2.5 mm and 5 mm from the tip over 120 s (PAPER.md:147,
 * Fig. 6 :250, Fig. 14 :282) and, per displayed frame, hands the finished buffer to the renderer while
 * the next iteration runs into the other one (Alg. 2). */

/* Set the probe points: n_probes flat voxel indices into the batched volume,
 * index = scenario*nx*ny*nz + i + nx*(j + ny*k)  (host array, copied; n_probes = 0 clears them). */
int rfa_set_probes(rfa_sim *s, int n_probes, const int64_t *index);

/* Advance n steps and record the probe temperatures (deg C) after every `every` steps:
 * out[m*n_probes + p] = T at probe p after (m+1)*every steps, m < n/every  (n must be a multiple of
 * every; every >= 1).  `out` is host or device memory of (n/every)*n_probes floats.  The stepping uses
 * the configured kernel (launches of up to fused_steps steps between records); the call returns after
 * the records have arrived in `out`. */
int rfa_step_record(rfa_sim *s, int n, int every, float *out);

/* rfa_step_record for callers that cannot allocate device memory when they call it.
 *
 * Why it exists: rfa_set_probes and rfa_step_record (host `out`) get the probe list and the row buffer from cudaMalloc, on
 * the first use and again whenever a longer series is asked for.  cudaMalloc / cudaFree wait for the whole GPU, so inside a
 * running frame loop (Alg. 2) they stall every stream of the device; and a host application that has handed the card's
 * memory to its own pool at start-up, or runs under a fixed memory budget, gets an error from them.  This call uses neither:
 * list and rows live in a fixed array inside the library image, RFA_STATIC_RECORD_MAX_PROBES * 8 +
 * RFA_STATIC_RECORD_MAX_FLOATS * 4 bytes (1 MiB + 8 KiB), which every GPU that loads librfa.so holds until the process ends.
 * It calls no cudaMalloc, cudaFree or other allocating routine.  (rfa_create allocates nothing on the device either when it
 * is given a workspace.)
 *
 *   n, every   as rfa_step_record: n time steps, one record after every `every` of them (n a multiple of every)
 *   n_probes   1 .. RFA_STATIC_RECORD_MAX_PROBES
 *   index      host, n_probes flat voxel indices (as rfa_set_probes); read before the call returns.  The list given to
 *              rfa_set_probes is neither used nor changed.
 *   out        host or device, (n/every)*n_probes floats, out[m*n_probes + p] = T (deg C) at probe p after (m+1)*every steps
 * Limits: n_probes > RFA_STATIC_RECORD_MAX_PROBES or (n/every)*n_probes > RFA_STATIC_RECORD_MAX_FLOATS -> RFA_E_INVALID
 * with both numbers in rfa_last_error(), nothing stepped; record a longer run as several calls.
 * Same kernels and same arithmetic as rfa_step_record: equal inputs give equal bits.  Returns after the records have arrived.
 *
 * Sharing: there is ONE such array per GPU for the whole process.  It keeps the previous call's contents (harmless: a call
 * overwrites every element it later reads, nothing has to start at zero), and two calls that run on the same GPU at the same
 * time -- from two host threads, on any simulations -- overwrite each other's rows.  The library takes no lock: serialise them.
 * First use: the first call on a GPU asks the CUDA runtime for the array's device address (once per device, kept afterwards).
 * Make that first call at start-up, before any stream capture is begun. */
enum { RFA_STATIC_RECORD_MAX_PROBES = 1024, RFA_STATIC_RECORD_MAX_FLOATS = 262144 };
int rfa_step_record_static(rfa_sim *s, int n, int every, int n_probes, const int64_t *index, float *out);

/* Frame hand-off (Alg. 2): device pointer of the finished image of one scenario as stored,
 * theta = T - t_blood (fp32, nx*ny*nz, x fastest), and t_blood.  The image stays untouched by the NEXT
 * launch of this simulation (it writes the other buffer) and is overwritten by the one after it: a
 * consumer on another stream may read it while one more rfa_step launch (<= fused_steps time steps)
 * runs.  The caller orders its read after the producing work (rfa_synchronize or a stream event). */
int rfa_current_frame(rfa_sim *s, int scenario, const float **theta_dev, float *t_blood_c);

/* ---- breathing-motion warp (Eq. 14) -----------------------
 * T(x_t) = T_ref(x_t + u^-1(x_t, t)): the temperature shown at position x_t of the moving anatomy is the
 * reference-frame temperature looked up through the (inverse) motion field of the current breathing phase.
 *   disp   host or device, 3*nx*ny*nz floats: the displacement field in MILLIMETRES as three volumes
 *          (u_x, then u_y, then u_z; each x fastest like every volume)
 *   scale  factor applied to the field (the breathing amplitude of the phase, "interpolated" :133)
 *   out    host or device, nx*ny*nz floats, deg C:
 *          out[v] = trilinear interpolation of the current temperature image of `scenario` at the position
 *          (voxel centre of v) + scale*disp[v], sample positions clamped to the volume of voxel centres.
 * Reads the simulation state, does not change it.  Waits for the stream unless both `disp` and `out` are device
 * memory (then it is asynchronous like rfa_step; rfa_synchronize orders the caller's read of `out`). */
int rfa_warp_temperature(rfa_sim *s, int scenario, const float *disp, float scale, float *out);

/* ---- headless view of the heat zone (Figs. 11-12) ----------------
 * The paper shows the ablation zone as the 42.5 C isotherm in its VR / fluoroscopy views.  No graphics API
 * is involved here: an orthographic ray-march written as plain CUDA arithmetic into a device (or host) buffer.
 *   Image plane through the volume centre c (mm), spanned by e1 = normalise(up x dir), e2 = dir x e1 (dir
 *   normalised first); pixel (px,py) has the offset u = (px-(W-1)/2)*pixel_mm along e1, v likewise along e2.
 *   Ray: p(m) = c + u e1 + v e2 + (-R + m*step_mm) dir, m = 0 .. floor(2R/step_mm), R = half the volume diagonal.
 *   A sample counts if it lies inside the box of voxel centres; there T is interpolated trilinearly.
 *   tmax[py*W+px]  = maximum of T over the ray's samples (t_blood if none lies inside)            [deg C]
 *   depth[py*W+px] = m*step_mm of the first sample with T >= iso_c, or -1 if there is none        [mm]
 * Outputs: host or device, W*H floats each (1 <= W*H <= 2^28); depth may be NULL.  Host images are staged in a
 * library-owned device buffer that grows on demand.  Reads the state only.  Synchronous. */
typedef struct rfa_view {
    float dir[3];      /* viewing direction (any non-zero length) */
    float up[3];       /* not parallel to dir */
    int width, height; /* pixels */
    float pixel_mm;    /* pixel spacing on the image plane */
    float step_mm;     /* sample spacing along the ray */
    float iso_c;       /* isotherm for the depth image, e.g. 42.5 or 60 (:37) */
} rfa_view;
int rfa_render_zone(rfa_sim *s, int scenario, const rfa_view *view, float *tmax, float *depth);

int rfa_synchronize(rfa_sim *s);
void rfa_destroy(rfa_sim *s);
const char *rfa_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* RFA_H */
