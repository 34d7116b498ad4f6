/*
 * jefi.h — C-ABI of libjefi: the B200-native hot path of JefiPIC (arXiv 2209.07944).
 *
 * One opaque context per simulation on one GPU.  It owns (1) a device ring buffer with the last H time steps
 * of the sources rho, J and their backward time differences, (2) the translation-invariant delay table of the
 * uniform grid, (3) scratch for the cell-sorted deposit.  The six calls of the PIC cycle are
 *
 *     jefi_deposit -> jefi_push_sources -> jefi_field_step -> jefi_push_particles
 *
 * Conventions common to every call
 *   - Plain C types only.  Unless a parameter says "host", array arguments are DEVICE pointers owned by the
 *     caller (e.g. torch tensors); the library never frees or keeps them.  The context owns everything it
 *     allocates and releases it in jefi_destroy.
 *   - Work is enqueued on the cudaStream_t given in jefi_config.stream (NULL = legacy default stream) and the
 *     call returns without synchronising, except where stated ("host" variants and debug exports synchronise).
 *   - Return value: 0 (JEFI_OK) or a negative JEFI_E* code; jefi_last_error() then returns a text.  No call
 *     aborts, throws or falls back to the CPU.
 *   - Grid: nx*ny*nz cuboid cells, cell index c = i + nx*(j + ny*k) (x fastest); every field lives at the cell
 *     centre ((i+.5)dx, (j+.5)dy, (k+.5)dz).  Sources and observation points share the grid.
 *   - Particles: positions in GRID UNITS (xi = x/dx in [0,nx), ...), momenta u = gamma*v/c (dimensionless).
 *     These are "flexible units" in the sense of PAPER.md:233 and make the cell index bit-exact.
 *   - Step counter n starts at -1; each jefi_push_sources makes it n+1 and stores the sources of step n.
 */
#ifndef JEFI_H
#define JEFI_H

#ifdef __cplusplus
extern "C" {
#endif

#define JEFI_OK 0
#define JEFI_EINVAL (-1) /* NULL / out-of-range argument */
#define JEFI_ENOMEM (-2) /* host or device allocation failed */
#define JEFI_ECUDA (-3)  /* a CUDA runtime call failed; text in jefi_last_error */
#define JEFI_ESTATE (-4) /* call not valid in this state (e.g. field_step before any push_sources) */

/* field_impl values */
#define JEFI_FIELD_AUTO 0      /* tiled kernel when its delay arithmetic is proven equal to the fp64 table, else reference;
                                  jefi_field_impl_reason() says which one runs and why */
#define JEFI_FIELD_REFERENCE 1 /* one thread per observation cell, table-driven delays (slow; the paper's K1 in fp32) */
#define JEFI_FIELD_TILED 2     /* shared-memory tiled kernel; jefi_create fails with JEFI_ESTATE if not provable */

/* field_tile values */
#define JEFI_TILE_AUTO 0
#define JEFI_TILE_CELL 1
#define JEFI_TILE_DYAD 2

/* deposit_mode values */
#define JEFI_DEPOSIT_AUTO 0   /* = JEFI_DEPOSIT_RUNS (the measured best on sorted and unsorted lists) */
#define JEFI_DEPOSIT_DIRECT 1 /* caller's order; lanes of a warp that hit the same node are combined wherever they sit (match-any) */
#define JEFI_DEPOSIT_SORTED 2 /* internal counting sort by cell (context scratch, every call), then JEFI_DEPOSIT_RUNS over that order */
#define JEFI_DEPOSIT_RUNS 3   /* caller's order; runs of neighbouring lanes in the same cell are combined before the fp32 reductions
                                 leave the SM: one reduction per (warp, cell, node, quantity) when the list is cell-sorted
                                 (jefi_sort_particles).  Two kernels do this (segmented shuffle reduction; transposition through
                                 shared memory, one 32-lane reduction per run); the context takes the first while the caller's
                                 list was sorted by jefi_sort_particles within the last 64 deposits, else the second
                                 (DESIGN.md section 6.3).  Same sums up to the order of the additions. */

/* delay_rule values: how the retarded time t_r = t^n - R/c of Eq. (2.6), which is not a stored step, is served */
#define JEFI_DELAY_NEAREST 0 /* sources and differences at the nearest stored step, m = floor(R/(c dt) + 1/2) (A1) */
#define JEFI_DELAY_LINEAR 1  /* same m and the same two samples; the VALUES rho, J are taken on the straight line through
                                them, S(t_r) = S^{n-m} - phi (S^{n-m} - S^{n-m-1}), phi = R/(c dt) - m in [-1/2, 1/2)
                                (second order in dt); the time derivatives stay (S^{n-m} - S^{n-m-1})/dt (A22) */

typedef struct jefi_ctx jefi_ctx; /* opaque */

typedef struct {
  int nx, ny, nz;       /* cells per axis (>= 1) */
  double dx, dy, dz;    /* cell size, metres (> 0) */
  double dt;            /* time step, seconds (> 0) */
  double c, eps0;       /* 0 -> SI values 299792458 and 8.8541878128e-12; mu0 := 1/(eps0 c^2) */
  int H;                /* ring depth in steps; 0 -> N_dt + 2 with N_dt = min(ceil(Lmax/(c dt)), hist_cap),
                           Lmax the diagonal of the region.  Delays m > H-2 contribute zero. */
  int hist_cap;         /* 0 -> 10000 */
  double Eext[3];       /* uniform background E, V/m, added at the particle */
  double Bext[3];       /* uniform background B, tesla */
  int device;           /* CUDA device ordinal */
  void* stream;         /* cudaStream_t; NULL -> default stream */
  int field_impl;       /* JEFI_FIELD_* */
  int deposit_mode;     /* JEFI_DEPOSIT_* */
  int delay_rule;       /* JEFI_DELAY_* */
  int shape_order;      /* particle shape function of jefi_deposit / jefi_push_particles: 0 or 1 -> S^(1), the linear (CIC,
                           volume-weighted) weights the paper uses, Eqs. (2.13), (2.16), (2.20); 2 -> S^(2), the quadratic
                           spline of Eq. (2.14) on 27 nodes (DESIGN.md section 3 A11) */
  int field_chunk;      /* tuning of the tiled field kernel: source tiles per CTA.  0 -> automatic (the range is
                           split over CTAs, into 32 pieces on large grids for L2 locality and to fill the GPU on small ones;
                           the partial sums, 24 N bytes per piece in context scratch, are added by a second kernel in a
                           fixed order); > 0 -> that many; -1 -> never split.
                           The result is deterministic (bit-identical from run to run) for every value. */
  int field_tile;       /* tuning of the tiled field kernel: what one thread of an observation tile owns.  0 -> automatic (dyads
                           once the grid has 32 tiles of 16x8x8 cells and nx pads no worse than with 8-wide tiles);
                           1 -> JEFI_TILE_CELL: one cell (8x8x8 tiles); 2 -> JEFI_TILE_DYAD: two cells that are neighbours along x
                           (16x8x8 tiles; needs nx >= 16): the pairs (r, r') and (r + ex, r' + ex) have the same offset, so their
                           distance, delay and geometric factors are evaluated once for both.  Ignored on nx <= 3 grids.  Every
                           choice forms the sums of Eqs. 2.4-2.5 over the same pairs; only the order of the additions differs. */
} jefi_config;

/* Fill *cfg with the defaults (every member zero, which each member documents as "automatic" / SI value / device 0 / legacy
 * stream) after checking that the caller's jefi_config has the size this library was built with: pass sizeof(jefi_config).
 * The struct carries no size or version member, so a program compiled against an older header (the struct has grown over
 * time, always at the end) would otherwise hand jefi_create uninitialised tail members.  Returns JEFI_OK, or JEFI_EINVAL if
 * cfg is NULL or sizeof_cfg differs (text through jefi_last_error(NULL)); *cfg is not touched in that case.  Never needs a GPU. */
int jefi_config_init(jefi_config* cfg, unsigned long sizeof_cfg);

/* Create a context: allocates the ring (32*H*N_padded bytes, zeroed = "zero before t0"), builds the
 * delay table m(|di|,|dj|,|dk|) = floor(R/(c dt) + 1/2) in fp64 on the host (Eq. 2.6; nearest-step reading,
 * DESIGN.md §3 A1) and verifies on the device that the tiled kernel's fp32 delay arithmetic reproduces it for
 * every offset.  *out is set to NULL on failure.  Synchronises. */
int jefi_create(const jefi_config* cfg, jefi_ctx** out);

/* Release everything the context owns.  NULL is a no-op.  Synchronises the context's stream first. */
void jefi_destroy(jefi_ctx* ctx);

/* Text of the last error of this context ("" if none).  ctx == NULL returns the last jefi_create error. */
const char* jefi_last_error(const jefi_ctx* ctx);

/* Values the context resolved at create time (H, N_dt, which field kernel runs ...).  All optional (NULL ok). */
int jefi_get_info(const jefi_ctx* ctx, int* H, int* ndt, int* field_impl, long* step, long* ring_bytes);

/* Why the context runs the field kernel it runs (one line of text, never NULL): e.g. "tiled: fp32 delays proven on 13824
 * offsets, window 36 slots in pitch 36, 1 pass" or "reference: 3 fp32 delay mismatches against the fp64 table". */
const char* jefi_field_impl_reason(const jefi_ctx* ctx);

/* Geometry of the tiled field kernel (all optional, NULL ok): observation tile and source tile in cells per axis
 * (8x8x8 or 16x8x8 / 4x4x4, see jefi_config.field_tile; 1x16x32 / 1x8x8 on grids with nx <= 3 such as the paper's 1 x ny x nz slabs), the largest slot window of a
 * tile pair, the shared-memory pitch it is served from (window > pitch: the tile is evaluated in ceil(window/pitch) passes),
 * and the number of pieces the source range is split into.  obs_tile[2] is the granularity of jefi_field_step_slab. */
int jefi_get_tile_info(const jefi_ctx* ctx, int obs_tile[3], int src_tile[3], int* window_slots, int* window_pitch,
                       int* source_split);

/* CIC (volume-weighted) charge/current deposit, Eqs. (2.15)-(2.19).
 *   np            number of macro-particles (>= 0)
 *   x,y,z         positions, grid units, np floats each
 *   ux,uy,uz      u = gamma v / c, np floats each; v = c u / sqrt(1+|u|^2)
 *   qw            charge of each macro-particle, coulomb
 *   alive         np bytes, 0 = dead (skipped); NULL = all alive
 *   rho,jx,jy,jz  OUT, N floats each (C/m^3, A/m^2), overwritten (zeroed by the call).
 * Node (i,j,k) = floor(xi-.5) ... gets q*w/dV with the 8 trilinear weights (shape_order 2: the 27 nodes around the
 * centre node floor(xi) with the S^(2) weights of Eq. 2.14); nodes outside the grid are virtual
 * and dropped.  Sums are fp32 atomics: the order of equal-cell particles is not defined.
 * The caller's particle arrays are never modified: with JEFI_DEPOSIT_SORTED the cell order is an index array in
 * context scratch (12 bytes per particle + 8 bytes per cell, allocated on first use).  np < 2^31. */
int jefi_deposit(jefi_ctx* ctx, long np, const float* x, const float* y, const float* z, const float* ux,
                 const float* uy, const float* uz, const float* qw, const unsigned char* alive, float* rho,
                 float* jx, float* jy, float* jz);

/* The cell-sorted deposit for callers that cannot allocate device memory.
 *
 * jefi_deposit in JEFI_DEPOSIT_SORTED mode keeps its sort scratch in the context and (re)allocates it with cudaMalloc on
 * first use and whenever np grows; creating the context allocates too.  That rules it out for a program whose device memory
 * is all owned by its own pool after start-up (no driver allocation may happen later, or would fail against its budget) and
 * for a step loop with a latency bound (cudaMalloc / cudaFree may synchronise the whole device).  This call needs no context
 * and calls no cudaMalloc, cudaFree or other allocating routine, on the first call or any later one: its scratch (sort key,
 * rank and order per particle, count and offset per sort bin, scan sums) is a fixed array of JEFI_STATIC_SCRATCH_BYTES
 * (16 MiB) inside the library's CUDA module, held by every GPU the library is loaded on until the process exits.
 *
 * Computes exactly what jefi_deposit computes with shape_order 1 (Eqs. 2.15-2.19; virtual nodes dropped,
 * PAPER.md:191; dead particles skipped), with the same kernels: same sums up to the order of the fp32 additions.
 *   device, stream   CUDA device ordinal (made current for the call, then restored) and the cudaStream_t (NULL = legacy default
 *                    stream) the work is enqueued on; the call does not synchronise
 *   nx,ny,nz,dx..dz  grid, as in jefi_config;  c: speed of light, 0 -> 299792458
 *   np, x..alive     as in jefi_deposit (DEVICE pointers, caller-owned, never modified; alive may be NULL)
 *   rho,jx,jy,jz     OUT, DEVICE, nx*ny*nz floats each, overwritten
 *   errbuf           HOST char[errbuf_len] that receives the text of an error (NULL / 0: no text)
 * Limits (the scratch cannot grow): np <= JEFI_STATIC_MAX_PARTICLES and (nx+1)(ny+1)(nz+1)+1 <= JEFI_STATIC_MAX_BINS, e.g. up
 * to a 79^3 grid.  Beyond either the call does nothing and returns JEFI_EINVAL with the limit named in errbuf; use jefi_deposit.
 * Set-up: the first call on each device looks up the device address of the scratch (cudaGetSymbolAddress; no allocation) and
 * caches it.  Make that first call per device before any stream capture begins.
 * Sharing: all calls on a device use the same array, and it keeps what the last call left.  The call itself clears the part
 * that must start at zero (the bin counters) on `stream` and overwrites the rest before reading it, so back-to-back calls on
 * ONE stream, with any mix of grids and list lengths, are independent.  Calls whose GPU work can overlap - different streams,
 * or different host threads - race on the array and give wrong sums: serialise them (one stream, or an event between them).
 * Returns JEFI_OK, JEFI_EINVAL (bad argument or over a limit) or JEFI_ECUDA. */
#define JEFI_STATIC_MAX_PARTICLES 1048576L
#define JEFI_STATIC_MAX_BINS 524288L
#define JEFI_STATIC_SCRATCH_BYTES 16781312L /* 3 x 4 MiB per-particle + 2 x 2 MiB per-bin + 4 KiB scan sums */
int jefi_deposit_static(int device, void* stream, int nx, int ny, int nz, double dx, double dy, double dz, double c, long np,
                        const float* x, const float* y, const float* z, const float* ux, const float* uy, const float* uz,
                        const float* qw, const unsigned char* alive, float* rho, float* jx, float* jy, float* jz, char* errbuf,
                        int errbuf_len);

/* Put the caller's particle arrays in cell order, in place: first the depositing particles (alive, at least one node
 * inside the grid) grouped by base node (i,j,k) = floor(xi-.5).. with i fastest, then all others.  The order inside a
 * group is not defined.  Optional for correctness (no call depends on the order), it is what makes the warp-level
 * combination of jefi_deposit and the field gathers of jefi_push_particles coalesce; particles move at most c dt per
 * step, so sorting every few steps is enough.  All of x..alive are IN/OUT np-element arrays; tag is an optional
 * (NULL ok) int array permuted along with them, e.g. particle ids.  Uses context scratch (53 bytes per particle). */
int jefi_sort_particles(jefi_ctx* ctx, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz,
                        float* qw, float* q_over_m, unsigned char* alive, int* tag);

/* Store the sources of the next step: n += 1, ring slot n mod H <- (rho, J) and their backward differences
 * against step n-1 (the finite differences of Eqs. 2.4-2.5; zero history before step 0).
 * rho,jx,jy,jz: N floats each, cell order x fastest. */
int jefi_push_sources(jefi_ctx* ctx, const float* rho, const float* jx, const float* jy, const float* jz);

/* Jefimenko field solve at the current step n, Eqs. (2.4)-(2.6), PAPER.md:103-109:
 *   E(r) =  dV/(4 pi eps0) sum_{r'!=r} [ d rho/R^3 + d rho_dot/(c R^2) - J_dot/(c^2 R) ]
 *   B(r) = -mu0 dV/(4 pi)  sum_{r'!=r} [ d x J/R^3 + d x J_dot/(c R^2) ]
 * with d = r - r', sources at step n - m(d), time derivatives from steps n-m and n-m-1, the self cell skipped
 * (PAPER.md:221).  ex..bz: OUT, N floats each (V/m, tesla), overwritten.
 * Sources before step 0 are zero: tile pairs all of whose delays reach back before step 0 are skipped, and so
 * are source tiles that held no charge or current during the steps a window reads (jefi_push_sources tracks that per tile).
 * The first steps of a run and mostly empty grids cost only what can contribute; results are identical, the skipped pairs
 * add exactly zero.
 * JEFI_ESTATE before the first jefi_push_sources. */
int jefi_field_step(jefi_ctx* ctx, float* ex, float* ey, float* ez, float* bx, float* by, float* bz);

/* The same solve restricted to the observation cells of the z-planes k0 <= k < k1 (all sources, as always): only those
 * entries of ex..bz are written.  Observation cells are independent (Eqs. 2.4-2.5 are sums per observation point), so
 * disjoint slabs computed by different calls - or by different GPUs that hold the same history, SURVEY.md §8(e) - add up to
 * jefi_field_step bit for bit (every sum is formed in a fixed order, also when the source range is split over CTAs).
 * k0 must be a multiple of the observation tile's z edge (jefi_get_tile_info: 8, or 32 on nx <= 3 grids); JEFI_EINVAL
 * otherwise. */
int jefi_field_step_slab(jefi_ctx* ctx, int k0, int k1, float* ex, float* ey, float* ez, float* bx, float* by, float* bz);

/* jefi_field_step that ALSO writes E, B interleaved per cell, eb_packed[8*c + 0..7] = (Ex, Ey, Ez, Bx, By, Bz, 0, 0) (DEVICE,
 * 8*N floats, 16-byte aligned): the layout jefi_push_particles_packed gathers from (two 16-byte loads per node instead of
 * six scattered words).  Written by the field kernel's own epilogue, no extra pass.  ex..bz as in jefi_field_step. */
int jefi_field_step_packed(jefi_ctx* ctx, float* ex, float* ey, float* ez, float* bx, float* by, float* bz, float* eb_packed);

/* Field interpolation (Eq. 2.20) + relativistic Boris push (Eqs. 2.7-2.11, DESIGN.md §3 A5/A6) + kill rule
 * (PAPER.md:205, 239): for each alive particle gather E,B from the 8 nodes (virtual nodes count as zero), add
 * Eext/Bext, update u and then the position by v*dt; a particle whose new position leaves [0,n) on any axis gets
 * alive = 0 and is never pushed or deposited again.
 *   x..uz   IN/OUT np floats each;  q_over_m  np floats (C/kg);  alive IN/OUT np bytes (must not be NULL)
 *   ex..bz  fields at step n, N floats each. */
int jefi_push_particles(jefi_ctx* ctx, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz,
                        const float* q_over_m, unsigned char* alive, const float* ex, const float* ey,
                        const float* ez, const float* bx, const float* by, const float* bz);

/* The same push reading the fields from the interleaved array jefi_field_step_packed wrote (8*N floats, DEVICE). */
int jefi_push_particles_packed(jefi_ctx* ctx, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz,
                               const float* q_over_m, unsigned char* alive, const float* eb_packed);

/* One whole PIC step n (PAPER.md:85 section 2, :231 section 2.4) in one call: jefi_deposit(r^n, u^{n-1/2}) -> jefi_push_sources ->
 * jefi_field_step_packed -> jefi_push_particles_packed, with the argument meanings of those calls (rho..jz: OUT, the deposited
 * sources of step n; ex..bz and eb_packed: OUT, the fields of step n; particle arrays IN/OUT).  When the context's stream is
 * not the legacy default stream, the sequence is captured into a CUDA graph on the first call (again whenever an argument
 * changes) and replayed as ONE launch afterwards: on small grids, where the kernels of a step take tens of microseconds, the
 * per-launch overhead is as large as the work.  The step counter lives on the device for the graph; it may be mixed freely with
 * the individual calls.  The graph is also captured afresh when context state it depends on changes: the sort scratch (grown by
 * another call with a longer list) or the run-deposit kernel JEFI_DEPOSIT_RUNS picks (it changes 64 deposits after the last
 * jefi_sort_particles; replays count as deposits).  On the legacy default stream (not capturable) the four calls are simply issued in turn. */
int jefi_pic_step(jefi_ctx* ctx, long np, float* x, float* y, float* z, float* ux, float* uy, float* uz, const float* qw,
                  const float* q_over_m, unsigned char* alive, float* rho, float* jx, float* jy, float* jz, float* ex, float* ey,
                  float* ez, float* bx, float* by, float* bz, float* eb_packed);

/* End-to-end variant of one field step with HOST buffers (pinned memory recommended): copies the newest source
 * slice (4 x N floats) host->device, does jefi_push_sources + jefi_field_step, copies E,B (6 x N floats)
 * device->host and synchronises the stream.  Host arrays: src_host = [rho|jx|jy|jz] (4N floats),
 * eb_host = [ex|ey|ez|bx|by|bz] (6N floats). */
int jefi_field_step_host(jefi_ctx* ctx, const float* src_host, float* eb_host);

/* Number of kernel launches this context has enqueued so far (bench.py's gpu_launches). */
long jefi_launch_count(const jefi_ctx* ctx);

/* Duration in milliseconds of the most recent jefi_field_step's main kernel, measured with CUDA events on the
 * context's stream.  Synchronises on the end event.  < 0 if no field step ran.  Steps that jefi_pic_step replays from its
 * CUDA graph record no events (a graph holds none): after such steps this still reports the last field step that was issued
 * directly (jefi_field_step*, or jefi_pic_step on the legacy default stream). */
float jefi_last_field_kernel_ms(jefi_ctx* ctx);

/* The same for the field step `calls_back` calls ago (0 = the most recent; the context keeps the events of its last 64
 * field steps), so that a timed loop can be read back afterwards without a synchronisation inside it.  < 0 if out of range. */
float jefi_field_kernel_ms(jefi_ctx* ctx, int calls_back);

/* ---- debug / parity exports (synchronise; not on the timed path) ---- */
/* The library's own memory checks.  A build with -DJEFI_CHECKED (libjefi_checked.so, `python -m paper_2209_07944_b200.build
 * --checked`) verifies on the device that every shared-memory address of the field kernel lies inside the rows staged for its
 * item [0], that pipeline stages are read in sequence [1], that the cell sort scatters inside the list [2], and poisons
 * stages with NaN before refilling them.  errors_host = HOST long[4] of violation counts since the library was loaded;
 * returns 1 in a checked build, 0 (JEFI_OK, counters always zero) in the normal one, < 0 on error.  Synchronises. */
int jefi_debug_check_errors(jefi_ctx* ctx, long errors_host[4]);
/* FP32 roofline probe: all SMs run independent register-resident FMA chains, timed with CUDA events on the context's stream;
 * *tflops_out = 2 * FMAs / time (HOST double), *sm_count_out the SM count (optional).  mode 0: scalar fma.rn.f32 whose
 * multiplier and addend are shared by all chains (the pipe itself); 1: the same with fma.rn.f32x2 (SASS FFMA2); 2 and 3: scalar /
 * packed chains in which every FMA reads three registers of its own (the register-file side of the pipe, which is what
 * bounds the field kernel).  Mode 0 is the measured denominator next to the derived
 * 148 x 128 x 2 x clock figure.  JEFI_EINVAL for any other mode. */
int jefi_debug_fp32_peak(jefi_ctx* ctx, int mode, double* tflops_out, int* sm_count_out);
/* Shared-memory delivery probe: SM cycles (at the maximum SM clock) one warp-wide LDS.128 costs the data pipe when the 32 lanes
 * read ring rows in a given pattern; 16 warps per SM issue nothing else.  pattern 0: all lanes one quad; 1: lane pairs
 * (2k, 2k+1) share a quad, 16 rows; 2: 32 rows; 3: as 1 but one pair differs; 4: as 1 with rows 8 slots apart inside a
 * half-warp (same 16-byte bank group).  *cycles_out is a HOST double.  This is the second roofline of the field kernel
 * (two LDS.128 per source-observation pair).  JEFI_EINVAL for any other pattern. */
int jefi_debug_lds128_cycles(jefi_ctx* ctx, int pattern, double* cycles_out);
/* m for every non-negative offset (a,b,c): m_out[a + nx*(b + ny*c)], HOST int array of N entries (SURVEY.md §8(b) sketched
 * short*; delays reach the history cap of 10000 and the device table is int, so int it is). */
int jefi_debug_delay_table(jefi_ctx* ctx, int* m_out_host);
/* Node index (i,j,k) = floor(xi - .5) of each particle as the deposit/push kernels compute it (shape_order 2: the centre
 * node floor(xi)): ijk_out = DEVICE int array [np][3]. */
int jefi_debug_cell_index(jefi_ctx* ctx, long np, const float* x, const float* y, const float* z, int* ijk_out);
/* The cell order that JEFI_DEPOSIT_SORTED and jefi_sort_particles use for these positions: order_out = DEVICE int
 * array [np], a permutation of 0..np-1 whose first *n_alive_host entries are the depositing particles grouped by base
 * node (i fastest, then j, then k); the order inside a group is not defined.  n_alive_host is a HOST long. */
int jefi_debug_cell_order(jefi_ctx* ctx, long np, const float* x, const float* y, const float* z,
                          const unsigned char* alive, int* order_out, long* n_alive_host);
/* The stored sources of step n - steps_back: out4N = DEVICE float array [4][N] = rho, Jx, Jy, Jz (J rescaled
 * back to A/m^2).  JEFI_EINVAL if that step is not in the ring. */
int jefi_debug_history_slot(jefi_ctx* ctx, int steps_back, float* out4N);

#ifdef __cplusplus
}
#endif
#endif /* JEFI_H */
