/*
 * gadep.h -- C ABI of the B200-native Gadep photon-transport hot path (libgadep.so).
 *
 * The calls follow the paper's statement of the problem (PAPER.md = arxiv 2605.25963, /root/reference/PAPER.md):
 *   DetMesh hands a vector of Triangle records -- vertices, normal, inside / outside material -- to Gadep in memory
 *   (sec 2.2.3); Gadep stores the facets in a BVH (sec 2.4.3), transports photons
 *   (photoelectric, Compton, pair production; sec 2.4.1; coherent added by BASELINE.json configs[1]),
 *   localises them on boundary crossings from the nearest facet ahead and its side materials (PAPER.md:191,
 *   sec 2.4.2) and scores deposited energy in the sensitive germanium into a pulse-height spectrum,
 *   from which the full-energy-peak efficiency is read (sec 3.2).
 *
 * Conventions
 *   - every call returns 0 (GADEP_OK) or a negative gadep_status; nothing throws or aborts;
 *     gadep_last_error() gives a text for the last failure on that context.
 *   - units: mm, MeV, 1/mm.  All device arithmetic is float32; tallies are integers.
 *   - pointers marked HOST are read/written by the CPU during the call and may be freed afterwards (the library
 *     copies).  Pointers marked HOST-or-DEVICE are classified with cudaPointerGetAttributes.
 *   - all device work is enqueued on the cudaStream_t given to gadep_create (0 = legacy default stream);
 *     calls synchronise that stream before returning unless stated otherwise.
 *   - one context per host thread; a context owns its device buffers until gadep_destroy.
 *   - there is no CPU fallback: without a CUDA device gadep_create fails with GADEP_E_CUDA.
 */
#ifndef GADEP_H
#define GADEP_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct gadep_ctx gadep_ctx;

typedef enum {
    GADEP_OK = 0,
    GADEP_E_NULL = -1,        /* null handle or null required pointer                                       */
    GADEP_E_ORDER = -2,       /* call order violated (e.g. run before materials / mesh / BVH / source)      */
    GADEP_E_ARG = -3,         /* argument out of range (sizes, energies, intensities, n_lines, n_bins ...)  */
    GADEP_E_NONFINITE = -4,   /* non-finite vertex coordinate                                               */
    GADEP_E_INDEX = -5,       /* vertex / surface / material index out of range                             */
    GADEP_E_DEGENERATE = -6,  /* zero-area triangle                                                         */
    GADEP_E_NOT_CLOSED = -7,  /* a surface is not a closed, edge-manifold, consistently oriented mesh       */
    GADEP_E_CUDA = -8,        /* CUDA runtime error; text in gadep_last_error                               */
    GADEP_E_NOMEM = -9
} gadep_status;

#define GADEP_MAT_KILL (-1)       /* side material id that terminates the photon (world boundary)           */
#define GADEP_FILTER_NONE (-2)    /* gadep_trace_rays: accept every facet                                   */
#define GADEP_MAX_LINES 64
#define GADEP_MAX_MATERIALS 16

/* per-history flags written by gadep_run_histories */
#define GADEP_F_ESCAPED 1u        /* some photon of the history left the geometry (no facet ahead, or KILL) */
#define GADEP_F_PEAK 2u           /* full-absorption history: all energy deposited in scoring material      */
#define GADEP_F_LEAK 4u           /* no facet ahead while inside a non-world material (float32 corner case): */
                                  /* the photon was localised again from its current point and went on      */
#define GADEP_F_NONSCORING 8u     /* some energy deposited outside the scoring material                     */
/* bits 8..15: line index; bits 16..31: number of interactions (saturating) */

int gadep_create(gadep_ctx **out, int device, void *cuda_stream);
void gadep_destroy(gadep_ctx *ctx);
const char *gadep_last_error(const gadep_ctx *ctx);

/*
 * Materials (PAPER.md:179 names the physics models; the tables here are the caller's data).
 *   mu            HOST float[n_mat][4][n_grid], linear attenuation 1/mm on the log grid
 *                 E_i = e_min * (e_max/e_min)^(i/(n_grid-1)); channel 0 photoelectric, 1 Compton, 2 coherent, 3 pair.
 *                 Channels 0-2 are interpolated log-log (an entry <= 0 makes the bracket 0), channel 3 linearly.
 *   is_scoring    HOST unsigned char[n_mat]; != 0 marks the sensitive volume (active Ge).
 * n_mat <= GADEP_MAX_MATERIALS, 2 <= n_grid <= 1024.  Photons below e_min deposit locally (cut-off).
 */
int gadep_set_materials(gadep_ctx *ctx, int n_mat, int n_grid, double e_min_mev, double e_max_mev, const float *mu,
                        const unsigned char *is_scoring);

/*
 * Mesh = the Triangle vector of PAPER.md:111.  Closed surfaces, nested or disjoint, facets wound so that
 * n = (v1-v0) x (v2-v0) (Eq. 5) points out of the enclosed volume.
 *   vertices      HOST float[n_vert][3]
 *   triangles     HOST int[n_tri][3] vertex indices
 *   tri_surface   HOST int[n_tri], surface index of each facet, in [0, n_surf)
 *   surf_inside / surf_outside   HOST int[n_surf] material id on the inner / outer side, or GADEP_MAT_KILL
 *   world_material  material where no facet lies ahead
 * Checks: finite vertices, index ranges, zero-area facets, and per surface that every directed edge is matched by
 * exactly one opposite edge (closed + oriented; the side-id rule of PAPER.md:191 is only valid then).  The arrays are
 * copied to the device first and checked there; a rejected mesh leaves the context without a mesh.
 * Invalidates a previously built BVH.
 */
int gadep_load_mesh(gadep_ctx *ctx, const float *vertices, int n_vert, const int *triangles, const int *tri_surface,
                    int n_tri, const int *surf_inside, const int *surf_outside, int n_surf, int world_material);

/* Builds the BVH over the facets on the GPU: binary LBVH -> uncompressed 4-wide nodes (default
 * traversal) and 8-wide nodes with 8-bit quantised child boxes (measured alternative), and the
 * facet-clearance grid beside it (flights that provably meet no facet need no traversal; same answers).
 * flags: 0, or one of the two below.  The grid's plane lists (cells near facets; 2 - 3 ms for 40 k facets, they pay on long
 * runs of volume sources) are made by the first gadep_run of >= 2e7 histories after the build (flags 0), with the build
 * (GADEP_BUILD_PLANE_LISTS) or never (GADEP_BUILD_NO_PLANE_LISTS).  No result depends on the choice.  Timed by bench.py;
 * the time of lists made by a run is added to last_build_ms. */
#define GADEP_BUILD_PLANE_LISTS 1
#define GADEP_BUILD_NO_PLANE_LISTS 2
int gadep_build_bvh(gadep_ctx *ctx, int flags);

/* Nodes the wavefront kernels and gadep_trace_rays traverse: 4 = uncompressed 4-wide nodes (128 bytes; the default),
 * 5 = the same four children with 8-bit quantised boxes (64 bytes), 8 = compressed 8-wide nodes (96 bytes).  All hold the
 * same facets in conservative boxes: the ray cast returns identical hits (tests: 1e6 rays against brute force, 6e7 rays
 * between the three).  Without a call the ray cast takes the 64-byte nodes on hierarchies of more than 256 MB (a node
 * visit is a fetch from HBM there: 14 % faster) and everything else the uncompressed ones. */
int gadep_set_bvh_width(gadep_ctx *ctx, int width);

#define GADEP_SRC_POINT 0
#define GADEP_SRC_VOLUME 1
#define GADEP_SRC_BEAM 2
typedef struct {
    int kind;                      /* GADEP_SRC_POINT (isotropic) | _VOLUME (isotropic) | _BEAM (pencil)        */
    float pos[3];                  /* point / beam origin                                                       */
    float dir[3];                  /* beam direction (unit)                                                     */
    float cyl_r, cyl_z0, cyl_z1;   /* volume: cylinder about the z axis                                         */
    float ex_r, ex_z0, ex_z1;      /* volume: excluded coaxial cylinder (Marinelli well); ex_r = 0 disables it  */
    int n_lines;                   /* 1 .. GADEP_MAX_LINES                                                      */
    const float *line_mev;         /* HOST float[n_lines], each within [e_min, e_max]                           */
    const float *line_intensity;   /* HOST float[n_lines], >= 0, not all zero                                   */
} gadep_source;
int gadep_set_source(gadep_ctx *ctx, const gadep_source *src);

/*
 * Batched geometries (the paper's calibration use-case: several detectors x 13
 * energies): the source set by gadep_set_source is replicated at n_copies translations, offsets HOST float[n_copies][3]
 * -- one per detector of a scene that holds the detectors side by side, each in its own closed world surface.  History
 * h is emitted from copy h mod n_copies; its line is counted under copy * n_lines + l in emitted[] / peak[] /
 * gadep_fepe / the per-history flags, so one gadep_run returns one FEPE curve per detector (the spectrum is their sum).
 * n_copies in 1..8 with n_copies * n_lines <= GADEP_MAX_LINES; n_copies = 1 restores the plain source (offsets may be
 * NULL).  gadep_set_source resets it.
 */
int gadep_set_source_copies(gadep_ctx *ctx, int n_copies, const float *offsets);

#define GADEP_RUN_ASYNC 1          /* do not synchronise the stream; spectrum must then be a DEVICE pointer     */
#define GADEP_RUN_ACCUMULATE 2     /* add to the context's tallies instead of starting from zero                */
#define GADEP_RUN_HISTORY_PER_THREAD 4  /* measurement: the plain one-history-per-thread kernel instead of the   */
                                   /* warp-resident wavefront kernel (same results, bit for bit)                */
#define GADEP_RUN_PERSISTENT_LANES 8    /* measurement: one history per lane with refill (same results)           */
#define GADEP_RUN_PARITY_LOCALISATION 16 /* the paper's reworked localisation: the material at the  */
                                   /* start and after every boundary crossing comes from parity counting over  */
                                   /* all facets ahead (history-per-thread kernel); the side ids only mark KILL */
#define GADEP_RUN_PARTIAL_XS 32     /* the paper's "partial cross-section method": one remaining    */
                                   /* optical depth per process instead of total-mu sampling + a selection draw  */
                                   /* (history-per-thread kernel; same distribution, different random streams)   */
#define GADEP_RUN_WARP_SPECIALISED 64 /* measurement: traversal and physics on separate warps of a block, registers moved */
                                   /* between them with setmaxnreg (same results, bit for bit)                     */
#define GADEP_RUN_BVH8 256          /* measurement / cross-check: the wavefront kernel traverses the compressed      */
                                   /* 8-wide nodes instead of the uncompressed 4-wide ones (same results, bit for bit) */
#define GADEP_RUN_ELECTRON_RANGE 128 /* SURVEY.md 8(f) NEXT-4 (coupled photon-electron physics): every   */
                                   /* energy deposit becomes one electron, a straight segment of the Katz-Penfold   */
                                   /* range in an isotropic direction (Philox stream 3), cut at the first facet of  */
                                   /* its material; the rest goes to the material behind it.  History-per-thread    */
                                   /* kernel; needs gadep_set_densities.  DESIGN.md reading R16.                    */
typedef struct {
    int n_bins;                    /* spectrum bins over [0, e_max_mev); one extra overflow slot follows        */
    float e_max_mev;
    unsigned long long first_history;  /* global index of the first history (RNG key; multi-GPU sharding)        */
    int flags;
} gadep_run_opts;

/*
 * Transports histories [first_history, first_history + n_histories) and writes the pulse-height spectrum.
 *   spectrum      HOST-or-DEVICE unsigned long long[n_bins + 1]; last slot = overflow; may be NULL.
 * Random numbers: Philox4x32-10, key = seed, counter = (history, draw/4, stream) -- results do not depend on
 * the launch configuration.  n_histories == 0 is valid and gives zeros.
 */
int gadep_run(gadep_ctx *ctx, unsigned long long n_histories, unsigned long long seed, const gadep_run_opts *opts,
              unsigned long long *spectrum);

/*
 * FEPE of one line from the last gadep_run: mode 0 = exact counters peak[l] / emitted[l];
 * mode 1 = read from the spectrum: (S[b] - (S[b-1] + S[b+1]) / 2) / emitted[l].  std_err = binomial. HOST outputs.
 */
int gadep_fepe(const gadep_ctx *ctx, int line, int mode, double *fepe, double *std_err);

/*
 * The whole tally block of the context, for the one exchange of a sharded run: n = gadep_tally_size()
 * = n_bins + 1 + 2 * GADEP_MAX_LINES words: spectrum[n_bins + 1], emitted[GADEP_MAX_LINES], peak[GADEP_MAX_LINES].
 * gadep_get_tallies copies it out (HOST-or-DEVICE; a DEVICE copy is stream-ordered and not synchronised);
 * gadep_set_tallies replaces it, so that gadep_fepe / gadep_get_counters / gadep_broaden read the reduced
 * counters after an all-reduce.  Both need a previous gadep_run on this context (it fixes n_bins).
 */
int gadep_tally_size(const gadep_ctx *ctx);
int gadep_get_tallies(gadep_ctx *ctx, unsigned long long *out);
int gadep_set_tallies(gadep_ctx *ctx, const unsigned long long *in);

/*
 * Detector-resolution broadening of the spectrum of the last gadep_run (the paper's spectra are
 * unbroadened, PAPER.md:253-259 reads the FEPE from exact peaks).  FWHM(E)^2 = fwhm_a + fwhm_b E + fwhm_c E^2 [MeV^2,
 * E in MeV]; every bin's counts are spread as a Gaussian centred on the bin middle.  out: HOST-or-DEVICE
 * double[n_bins + 1]; bin 0 also takes the mass below 0, the last slot the overflow counts and the mass above e_max,
 * so the total is conserved.
 */
int gadep_broaden(gadep_ctx *ctx, double fwhm_a, double fwhm_b, double fwhm_c, double *out);

/* ---- test / measurement hooks ------------------------------------------------------------------------------ */

/*
 * Nearest facet along each ray through the BVH.  org, dir: HOST-or-DEVICE float[n_rays][3];
 * tri_out int[n_rays] (caller's triangle index, -1 = none) and t_out float[n_rays] in the same memory space.
 * filter_material: GADEP_FILTER_NONE, or accept only facets whose from-side material equals it.
 * t_min: hits need t > t_min (may be negative).
 */
int gadep_trace_rays(gadep_ctx *ctx, const float *org, const float *dir, long long n_rays, int filter_material,
                     float t_min, int *tri_out, float *t_out);

/*
 * gadep_trace_rays for callers that must not allocate (CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same nearest-facet query through the same traversal kernel, with every byte of
 * scratch -- the kernel's ray-fetch counter, its work counters and, for HOST arrays, the staging copies of org / dir /
 * tri_out / t_out (32 B per ray) -- in ONE file-scope `static __device__` array of the library
 * (256 + 256 + 32 * GADEP_STATIC_MAX_RAYS bytes = 8 MiB + 512 B, held by every GPU that loads the library until the
 * process exits).  Calls no cudaMalloc / cudaFree and no allocating library routine.
 *   org, dir, tri_out, t_out   as gadep_trace_rays (HOST or DEVICE, all in one memory space); the caller owns them
 *   n_rays                     0 .. GADEP_STATIC_MAX_RAYS; more -> GADEP_E_ARG ("... exceeds GADEP_STATIC_MAX_RAYS")
 * The array is shared by every context and every call on a device and keeps the previous call's contents: the entry
 * point clears the counters it needs at zero on the context's stream before the launch, and returns after the stream
 * has drained.  Two calls that overlap on the GPU (two contexts / streams / host threads on the same device) RACE on it;
 * serialise them.  The first call on a device resolves the array's device address (cudaGetSymbolAddress, which may load
 * the module); make that call outside a capture.  Work counters of the call: gadep_get_counters, as for gadep_trace_rays.
 */
#define GADEP_STATIC_MAX_RAYS (1 << 18)
int gadep_trace_rays_static(gadep_ctx *ctx, const float *org, const float *dir, long long n_rays, int filter_material,
                            float t_min, int *tri_out, float *t_out);

/*
 * Material in which each point lies (sec 2.4.2), found from a ray cast along dir.
 *   mode GADEP_LOCATE_SIDE_ID  the paper's original rule: nearest facet ahead; its normal tells entering from leaving and
 *                              the facet's side ids give the material (what gadep_run uses).
 *   mode GADEP_LOCATE_PARITY   the paper's reworked rule: intersections with every closed surface are counted (all-hits
 *                              BVH traversal); among the surfaces with an odd count the one whose first intersection
 *                              is nearest contains the point and its inside material is returned; none -> world.
 * org, dir: HOST-or-DEVICE float[n][3]; material_out int[n] in the same memory space.  A ray that meets more than 96
 * facets returns GADEP_LOCATE_OVERFLOW (-3) in parity mode.  Counters (box / triangle tests) as for gadep_trace_rays.
 */
#define GADEP_LOCATE_SIDE_ID 0
#define GADEP_LOCATE_PARITY 1
#define GADEP_LOCATE_OVERFLOW (-3)
int gadep_locate(gadep_ctx *ctx, const float *org, const float *dir, long long n, int mode, int *material_out);

/*
 * Densities of the materials [g/cm^3], HOST float[n_mat] (n_mat as in gadep_set_materials); used only by
 * GADEP_RUN_ELECTRON_RANGE to turn the Katz-Penfold range (mg/cm^2) into millimetres.  0 = no electron transport there.
 */
int gadep_set_densities(gadep_ctx *ctx, int n_mat, const float *rho_g_cm3);

/* Per-history dump (same arithmetic as gadep_run): edep_out float[n] scoring deposit (line energy for
 * full-absorption histories), flags_out unsigned[n] (GADEP_F_*).  HOST-or-DEVICE, either may be NULL. */
int gadep_run_histories(gadep_ctx *ctx, unsigned long long first, long long n, unsigned long long seed,
                        float *edep_out, unsigned *flags_out);
/* The same with the kernel-selecting GADEP_RUN_* flags of gadep_run (ASYNC and ACCUMULATE are ignored). */
int gadep_run_histories_ex(gadep_ctx *ctx, unsigned long long first, long long n, unsigned long long seed,
                           int run_flags, float *edep_out, unsigned *flags_out);

typedef struct {
    unsigned long long n_histories, n_queries, n_box_tests, n_tri_tests, n_crossings, n_pe, n_compton, n_coherent,
        n_pair, n_escaped, n_leak, n_cutoff;
    unsigned long long emitted[GADEP_MAX_LINES], peak[GADEP_MAX_LINES];
    int n_lines;
    int n_bvh_nodes, bvh_max_depth;
    float last_run_ms, last_build_ms;      /* CUDA-event times of the last gadep_run / gadep_build_bvh kernels   */
    int last_run_launches, last_build_launches;
    unsigned long long n_skipped_queries;  /* flights that end before the clearance of their grid cell: answered     */
                                           /* ("no facet") without a BVH query; n_queries counts only BVH queries     */
    unsigned long long n_stack_overflow;   /* rays that ran out of traversal stack since gadep_create (must be 0; a  */
                                           /* run that sees one fails with GADEP_E_ARG)                              */
    unsigned long long n_parity_queries;   /* GADEP_RUN_PARITY_LOCALISATION: all-hits localisation queries       */
    unsigned long long n_parity_mismatch;  /* ... of which the parity rule and the side ids named different media */
    unsigned n_grid_list_cells;            /* clearance grid: cells near facets (scalar bound below the lists' reach) ...  */
    unsigned n_grid_lists;                 /* ... of which got a plane list (0 = no lists made since the last build)      */
} gadep_counters;
/* Counters of the last gadep_run / gadep_run_histories / gadep_trace_rays (HOST output). */
int gadep_get_counters(const gadep_ctx *ctx, gadep_counters *out);

/* Raw Philox4x32-10 block from the device implementation (RNG pin against cuRAND's device routine):
 * which = 0 this library's generator, 1 = curand_Philox4x32_10 from <curand_philox4x32_x.h>.  HOST arrays. */
int gadep_philox_raw(gadep_ctx *ctx, const unsigned *ctr4, const unsigned *key2, int which, unsigned *out4);

#ifdef __cplusplus
}
#endif
#endif /* GADEP_H */
