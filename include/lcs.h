/*
 * lcs.h -- C ABI of liblcs_b200: the particle hot path of LCS.jl (arxiv/paper_2604_11008) on one
 * NVIDIA B200 (sm_100a).  Lagrangian step (trilinear gather, drag + gravity advance, 27-way
 * classification) followed by the prefix-scan particle communication among P = Px*Py*Pz virtual
 * subdomains held in one GPU's HBM.
 *
 * Citations: PAPER.md:<line> is /root/reference/PAPER.md (the only reference file); "DESIGN R-n"
 * is a numbered reading in DESIGN.md section 3 where the paper is silent or ambiguous.
 *
 * Conventions
 *  - Box: periodic cube [0, L)^3, L = 2*pi as the double 0x401921FB54442D18 (PAPER.md:47, L0 = 1).
 *  - Fluid: three N^3 fp64 arrays u,v,w at cell centres ((i+1/2)dx, ...), flat index
 *    i + N*(j + N*k), x fastest (DESIGN R-8).
 *  - Subdomain s = px + Px*(py + Py*pz); destination code c = (dx+1) + 3*(dy+1) + 9*(dz+1),
 *    d* in {-1,0,+1}, 13 = stay (DESIGN R-13).
 *  - Particle state: 8 SoA arrays x,y,z,vx,vy,vz,d (fp64) and id (int64)  (PAPER.md:150-162 lists
 *    17 Float64 arrays for two RK2 stages; a single stage needs these 8, DESIGN R-2).
 *  - Every d_* pointer is DEVICE memory owned by the caller, 16-byte aligned.  h_* pointers are
 *    HOST memory (pinned for full speed).  The library never allocates device memory: it carves
 *    the caller's workspace.  All calls enqueue on the handle's CUDA stream and return without
 *    synchronising unless stated.
 *  - Return value: 0 = LCS_OK, negative = error found on the host at call time.  Errors found on
 *    the device are sticky in a status word that lcs_get_status reads (capacity overflow, a
 *    particle that moved more than one subdomain or became non-finite, an input position outside
 *    [0,L)).  After a sticky error memory safety still holds and particle contents are unspecified.
 *    The calls never synchronise, so the host learns of a sticky error only through lcs_get_status:
 *    once lcs_get_status has returned it, every further stepping call (lcs_particle_step,
 *    lcs_migrate, lcs_migrate_sweeps, lcs_step_fused, lcs_step_rk2, lcs_step_fused_host) returns
 *    that code without doing work, until lcs_set_particles loads a fresh particle set.  A caller
 *    that never polls keeps stepping on unspecified contents.  (The paper is silent on errors:
 *    DESIGN R-16/17.)
 */
#ifndef LCS_B200_H
#define LCS_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LCS_OK                0
#define LCS_ERR_INVALID_ARG  (-1)
#define LCS_ERR_STATE        (-2)
#define LCS_ERR_CUDA         (-3)
#define LCS_ERR_CAPACITY     (-4)   /* sticky: a receiver slab or a send region overflowed        */
#define LCS_ERR_JUMP         (-5)   /* sticky: displacement > one subdomain, or non-finite        */
#define LCS_ERR_RANGE        (-6)   /* sticky: lcs_set_particles saw a position outside [0, L)     */
#define LCS_ERR_NOMEM        (-7)   /* host memory for the handle could not be allocated           */
#define LCS_ERR_TOO_LARGE    (-8)   /* lcs_pair_count_static: the handle exceeds the built-in scratch */

#define LCS_STAY_CODE 13

typedef struct lcs_handle lcs_t;    /* opaque, host memory, owned by the library */

/* Physical parameters, copied at create. */
typedef struct {
    double  nu;             /* kinematic viscosity, 1.5e-5 m^2/s                     */
    double  rho_ratio;      /* rho_p / rho: 843 in PAPER.md:57, 1000 in BASELINE.json's configs     */
    double  g[3];           /* gravity; (0,0,0) reproduces Eq. 6, DESIGN R-4          */
    int64_t send_capacity;  /* migrant slots per subdomain send region; 0 = capacity (never full)  */
    int32_t drag_model;     /* 0: Stokes drag, f = 1 (the hot path of BASELINE.json's configs);
                               1: f = 1 + 0.15 Re_p^0.687, Re_p = d|V-U|/nu (Eq. 7-8),
                                  frozen at the start of the step, tau_eff = tau_p / f (DESIGN R-23)  */
    int32_t enable_rk2;     /* 1: reserve the extra arrays of the paper's two-stage RK2 in the workspace (one group of 8
                               arrays of P*capacity doubles: X0, K1 and two spare) so that lcs_step_rk2 can be called */
} lcs_params;

/* Bytes of device workspace lcs_create needs; 0 if the arguments are invalid. */
size_t lcs_workspace_bytes(int N, int Px, int Py, int Pz, int64_t capacity, const lcs_params* prm);

/* Create a handle.  N: fluid grid points per axis (N >= 2, divisible by Px, Py and Pz, and
 * Px*Py*Pz*(N/Px+2)*(N/Py+2)*(N/Pz+2) < 2^32: the fluid is kept as one brick of cells plus a one-cell periodic halo
 * per subdomain and record indices are 32-bit, which allows N <= 1623 with one subdomain and less with many);
 * Px, Py, Pz: 1..1024 each, Px*Py*Pz <= 8192; capacity: particle slots per subdomain slab (it must
 * be even, so that slab bases and tile runs stay 16-byte aligned, and P*capacity < 2^31: slots are
 * 32-bit indices); LCS_ERR_INVALID_ARG otherwise.  d_workspace: device block of at
 * least lcs_workspace_bytes(), 256-byte aligned, borrowed until lcs_destroy; cuda_stream: a
 * cudaStream_t (NULL = legacy default stream). */
int lcs_create(int N, int Px, int Py, int Pz, int64_t capacity, const lcs_params* prm,
               void* d_workspace, size_t workspace_bytes, void* cuda_stream, lcs_t** out);
int lcs_destroy(lcs_t* h);

/* Fluid velocity on the N^3 cell centres, x fastest: u[i + N*(j + N*k)].  The three arrays are read
 * once, at call time in stream order, and repacked into the workspace as one 32-byte (u,v,w,0) record per cell (one
 * L2 sector per stencil corner), one contiguous brick of cells plus a periodic halo of one cell per subdomain -- what a
 * rank of the paper's decomposition holds; the caller may reuse them once the call's work has run.
 * LCS_ERR_INVALID_ARG for a null pointer or one that is not 16-byte aligned. */
int lcs_set_fluid(lcs_t* h, const double* d_u, const double* d_v, const double* d_w);

/* Load n particles given in any order; they are binned stably (input order kept inside each
 * slab) into the subdomain that contains them, all codes = stay.  Copies.  Positions must lie in
 * [0, L) (else sticky LCS_ERR_RANGE); a slab that would exceed capacity -> sticky LCS_ERR_CAPACITY.
 * LCS_ERR_INVALID_ARG for n < 0, n > P*capacity, a null pointer (n > 0) or one that is not 16-byte
 * aligned.  PAPER.md:47 (3-D decomposition), DESIGN R-12. */
int lcs_set_particles(lcs_t* h, int64_t n, const double* d_x, const double* d_y, const double* d_z,
                      const double* d_vx, const double* d_vy, const double* d_vz,
                      const double* d_diam, const int64_t* d_id);

/* a1-a4: per particle, interpolate U at X (trilinear), advance V then X under
 * dV/dt = -(V-U)/tau_p + g, dX/dt = V with U frozen over dt (Eq. 5-6, f = 1;
 * exponential integrator, DESIGN R-1), wrap into the box, classify into one of 27 destinations
 * ("mask computation") and count per (subdomain, destination).  In place.
 * LCS_ERR_STATE without fluid or particles, or while the codes of an earlier lcs_particle_step
 * are still waiting for lcs_migrate / lcs_migrate_sweeps (the same holds for lcs_step_fused and
 * lcs_step_rk2: a pending push must be migrated first). */
int lcs_particle_step(lcs_t* h, double dt);

/* a5-a8: prefix-scan particle communication among the virtual
 * subdomains, consuming the codes of the last lcs_particle_step: exclusive prefix scan of the
 * per-(subdomain, destination) indicator (single-pass decoupled look-back), stable pack of the
 * migrants, in-place stable compaction of the stayers, append in fixed order: receiver r holds
 * its stayers in original order, then incoming segments by (source s, code c, source slot)
 * ascending (DESIGN R-12).  LCS_ERR_STATE if no lcs_particle_step preceded it. */
int lcs_migrate(lcs_t* h);

/* The paper's own integrator: explicit two-stage RK2 (Heun) with one particle communication per stage (PAPER.md:64,
 * :150-164, :175-177; R-25).  Stage 1: K1 = (U(X0)-V0)/tau + g, X1 = X0 + dt V0, V1 = V0 + dt K1; X0, V0, K1 are
 * kept, everything live between the stages migrates (the paper's 17 arrays; here V1 is recomputed, so 14 + 2 spare).  Stage 2: K2 = (U(X1)-V1)/tau + g, X = X0 + dt/2 (V0+V1),
 * V = V0 + dt/2 (K1+K2); migrate.  tau = tau_p / f with f at the start of each stage (drag_model).  Explicit: meant for
 * dt/tau_p <= 0.5 (the paper's regime); BASELINE.json's configs need lcs_step_fused.  Needs lcs_params.enable_rk2 = 1
 * (LCS_ERR_STATE otherwise).  lcs_get_status then reports the migrants of the second migration. */
int lcs_step_rk2(lcs_t* h, double dt);

/* Axis-by-axis exchange (R-24): three sweeps x, y, z.  Each sweep classifies
 * every particle along one axis from its CURRENT position relative to the slab it sits in (minimum-image difference of
 * subdomain indices) and migrates with the three codes of that axis, in the order of lcs_migrate within the sweep.
 * After the call every particle is in the slab that contains it -- the same slab contents as lcs_migrate delivers, in the
 * sweeps' own (unique, deterministic) order.  May follow lcs_particle_step instead of lcs_migrate, or be called on its
 * own.  lcs_get_status then reports the migrants of the LAST sweep.  LCS_ERR_STATE without particles; a particle more
 * than one subdomain away from its slab along an axis raises the sticky LCS_ERR_JUMP. */
int lcs_migrate_sweeps(lcs_t* h);

/* lcs_particle_step followed by lcs_migrate in one pass that reads and writes each particle
 * once; the result is bit-identical to the two calls. */
int lcs_step_fused(lcs_t* h, double dt);

/* Per-subdomain particle counts, P int64 values, device pointer. */
int lcs_get_counts(lcs_t* h, int64_t* d_counts);

/* Packed copy-out: subdomain 0's particles in slot order, then subdomain 1's, ...  Each array
 * needs room for the current total (lcs_get_status gives it; <= P*capacity).  Any of the data
 * pointers may be NULL to skip that field; the others must be 16-byte aligned (LCS_ERR_INVALID_ARG). */
int lcs_get_particles(lcs_t* h, int64_t* d_counts, double* d_x, double* d_y, double* d_z,
                      double* d_vx, double* d_vy, double* d_vz, double* d_diam, int64_t* d_id);

/* Destination codes of the last lcs_particle_step in the same packed order (uint8, 13 after a
 * migrate); the P*27 count table (int64, row s, column c).  Test / diagnostic accessors. */
int lcs_get_codes(lcs_t* h, uint8_t* d_codes);
int lcs_get_count_table(lcs_t* h, int64_t* d_table);

/* Statistics hook: the pair count behind the radial distribution function g(r) ("radial distribution
 * function at contact g(r=R) ... unity indicates a uniform distribution"; the statistic the paper's heterogeneous run
 * offloads to a GPU; R-26).  Writes to *d_count (device, int64, 8-byte aligned) the number
 * of unordered pairs of ALL particles in the box whose periodic (minimum-image) separation r satisfies
 * r_lo <= r < r_hi; g over the shell = count / (n (n-1) / 2 * 4/3 pi (r_hi^3 - r_lo^3) / L^3).  Arithmetic per pair as
 * DESIGN.md R-26 fixes it, so the count is bit-exact against the O(n^2) definition.  Uses the send pool as scratch
 * (slot indices sorted by cell + a cell list of up to 256^3 cells): call it between steps, not between
 * lcs_particle_step and lcs_migrate.  LCS_ERR_INVALID_ARG unless 0 <= r_lo < r_hi <= L/3, and also when the send pool
 * cannot hold the scratch: it needs three arrays of P*capacity doubles plus at least 1 KB of cell list, i.e.
 * lcs_params.send_capacity of roughly 3/8 of capacity or more (0 = capacity always suffices); a handle with a smaller
 * pool can use lcs_pair_count_static below.  LCS_ERR_STATE without particles or with a pending push. */
int lcs_pair_count(lcs_t* h, double r_lo, double r_hi, int64_t* d_count);

/* lcs_pair_count for callers that have no device memory left to lend and may not ask the CUDA runtime for more.
 *
 * Who that is: lcs_pair_count borrows the handle's send pool for the positions sorted by cell and for its cell list,
 * and gives up (LCS_ERR_INVALID_ARG) when that pool is smaller than three position arrays -- which is exactly what a
 * production run has when it sized send_capacity for the few per cent of particles that migrate.  The obvious way out,
 * a larger workspace, is closed to a diagnostics hook that is called from inside a running time loop: by then the host
 * application (the flow solver, an in-situ analysis framework, a job that handed all of HBM to its own pool at start-up)
 * owns every byte of device memory and forbids cudaMalloc / cudaFree in the loop, because those calls stall every stream
 * of the device while they run and can fail with the memory already spoken for.  Such a caller passes what it has -- the
 * handle (its particles are the input) and the 8-byte result word -- and this entry point brings its own scratch.
 *
 * Where the scratch lives: in ONE array of LCS_PAIR_COUNT_STATIC_BYTES (17 MiB) that is part of the library's device
 * image.  Every GPU on which the library's kernels are loaded carries these 17 MiB from then until the process exits,
 * whether or not this function is ever called; that is the price, and the reason the limit is modest.  The call itself
 * performs no cudaMalloc, cudaFree or any other allocating runtime or library call, on the host or on the device.
 *
 * Limit: Px*Py*Pz*capacity <= LCS_PAIR_COUNT_STATIC_MAX_SLOTS (2^19 = 524,288 particle slots).  A larger handle gets
 * LCS_ERR_TOO_LARGE and nothing is enqueued: use lcs_pair_count with a send pool of at least 3/8 of capacity instead.
 *
 * First call on a device: looks up the device address of the array (cudaGetSymbolAddress with that device current) and
 * remembers it per device; later calls on that device only read the remembered pointer.  Make this first call during
 * set-up, outside any stream capture.  The device that is current at the call must be the one that owns the handle's
 * workspace (LCS_ERR_INVALID_ARG otherwise: each GPU has its own copy of the array, and another GPU's address is not
 * usable); with more than LCS_PAIR_COUNT_STATIC_MAX_DEVICES (64) devices, ordinals beyond that get LCS_ERR_INVALID_ARG.
 *
 * Sharing: all handles and all threads of the process that use one GPU share the one array.  It still holds the previous
 * call's cell list and sorted positions when a call begins; the call clears the part that has to start at zero (the cell
 * counters) in stream order before it uses it, so back-to-back calls on one stream are independent.  Two calls whose
 * GPU work can overlap -- different streams, or different host threads driving different handles -- race on the array
 * and both results are then garbage: serialise them (one stream, or an event between them).
 *
 * Same arguments, same result (bit-exact count), same state rules and error codes as lcs_pair_count otherwise; the send
 * pool is not touched, so unlike lcs_pair_count it does not matter how small send_capacity is. */
#define LCS_PAIR_COUNT_STATIC_MAX_SLOTS   (1 << 19)
#define LCS_PAIR_COUNT_STATIC_BYTES       (17u << 20)
#define LCS_PAIR_COUNT_STATIC_MAX_DEVICES 64
int lcs_pair_count_static(lcs_t* h, double r_lo, double r_hi, int64_t* d_count);

/* Synchronises the stream and reads the status word.  Any out pointer may be NULL.
 * Returns the sticky error (0 if none). */
int lcs_get_status(lcs_t* h, int* sticky_error, int64_t* n_total, int64_t* n_migrated_last);

/* End-to-end convenience with HOST buffers (what a CPU-resident caller pays; cf. the paper's
 * CPU-delegated path): copies n particles host->device, bins them, runs
 * lcs_step_fused(dt), copies the packed result and the P counts device->host, synchronises.
 * h_in / h_out: 8 host pointers each in the order x,y,z,vx,vy,vz,d,id (8 bytes per element;
 * h_out arrays need room for n; 8-byte aligned).  d_staging: device scratch, 256-byte aligned, of at
 * least lcs_staging_bytes(n, P) bytes (eight arrays of n words, each rounded up to 256 bytes, plus
 * the P counts; 0 for n < 0 or P < 1).  LCS_ERR_INVALID_ARG for a null or misaligned pointer or a
 * staging block that is too small.  The host copies run on a copy stream the handle creates on first use (the only CUDA
 * object the library creates besides profiling events; destroyed by lcs_destroy), ordered against the handle's stream by
 * events, one array at a time; host buffers should be pinned, or the copies serialise with the kernels.  On return the
 * handle's stream is synchronised and h_out / h_counts are complete. */
size_t lcs_staging_bytes(int64_t n, int P);
int lcs_step_fused_host(lcs_t* h, double dt, int64_t n, const void* const h_in[8], void* const h_out[8],
                        int64_t* h_counts, void* d_staging, size_t staging_bytes);

/* Optional per-kernel timing for benchmarks.  lcs_profile_begin creates CUDA events (no device
 * memory) and makes every following lcs_step_fused / lcs_migrate record four of them on the
 * handle's stream: before the tile pass, after it, after the table scan, after unpack + commit.
 * At most max_steps steps are recorded; later steps run untimed.  A "step" here is one migration round: lcs_step_rk2
 * records three (stage 1, the X0/K1 group, stage 2) and lcs_migrate_sweeps three (x, y, z), and n_steps counts them so.  lcs_profile_end synchronises the
 * stream, returns the summed durations in milliseconds and the number of recorded steps, and
 * destroys the events.  Any out pointer may be NULL. */
int lcs_profile_begin(lcs_t* h, int max_steps);
int lcs_profile_end(lcs_t* h, double* ms_tile_pass, double* ms_table, double* ms_unpack, int* n_steps);

/* (The only export that is not part of the path: a measurement aid, used by bench.py's roofline.l2_to_sm.)
 * Measurement aid for the roofline of the gather (a1): runs, alone on the handle's stream, a kernel in which every
 * lane issues eight independent 32-byte record loads per iteration (the gather's own load instruction, 12 warps per
 * SM) at pseudo-random records inside the first window_mb megabytes of the repacked fluid field, `iters` times, and
 * times it with CUDA events (synchronises).  *h_ms: duration in milliseconds, *h_bytes: sector bytes requested (host
 * pointers).  With a window that fits L2 (like one subdomain's brick) h_bytes / h_ms is the L2 -> SM ceiling of the
 * gather's access pattern on this GPU; with the whole field it is the DRAM random-sector rate.  Computes nothing that
 * the path uses.  LCS_ERR_STATE before lcs_set_fluid. */
int lcs_probe_gather(lcs_t* h, double window_mb, int iters, double* h_ms, double* h_bytes);

/* Number of kernels this library has launched on the handle since create (for bench accounting). */
int64_t lcs_kernel_launches(lcs_t* h);

/* Library build information: "lcs_b200 <version> sm_100a".  There are no ablation or debug builds of this library:
 * the kernels have no compile-time switches that change results. */
const char* lcs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* LCS_B200_H */
