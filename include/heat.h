/*
 * heat.h -- C-ABI boundary of the B200-native hot path of arXiv 1408.5853
 * (Ayriyan, Busa Jr., Donets, Grigorian, Pribis: "Algorithm and Simulation of Heat
 * Conduction Process for Design of a Thin Multilayer Technical Device").
 *
 * The library advances the paper's explicit-implicit finite-difference scheme, eq. (8)
 * P:L108-113 ("P:Lnnn" = line of the paper text), one time step T -> T^ at a time:
 *
 *     rho c_V(T) (T^ - T)/tau = Lambda_i[T^] + Lambda_j[T] + X        (8)
 *
 * implicit in r (one tridiagonal system per z-line, eqs. (12)-(20) P:L131-192), explicit in
 * z (eq. (11)), coefficients at the current level, no iterations.  All
 * arithmetic is fp64 and runs in hand-written sm_100a CUDA kernels; there is no CPU path.
 *
 * Conventions
 *   - i = radial node index 0..nr-1, j = axial node index 0..nz-1; node counts include the
 *     boundary nodes (nr = N+1, nz = M+1 in the paper's ranges, eq. (9)).
 *   - Field layout at this boundary: [batch][nz][nr], r fastest, fp64.
 *   - "host" / "device" is stated for every pointer.  The library never allocates device
 *     memory: the caller owns the two field levels, the workspace and the probe buffer and
 *     must keep them alive until heat_destroy.  Small host arrays are copied at create time.
 *   - Every call returns a heat_status; nothing throws or longjmps across the boundary.
 *     A message for the last failure is available from heat_last_error.
 *   - heat_step is asynchronous on the caller's stream; a CUDA fault raised by it surfaces
 *     as HEAT_ECUDA from the next synchronising call (heat_get_field to host, heat_probe).
 */
#ifndef HEAT_B200_H
#define HEAT_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct heat_ctx heat_ctx; /* opaque, owned by the library */

typedef enum {
    HEAT_OK = 0,
    HEAT_EINVAL = 1, /* malformed descriptor / argument */
    HEAT_ENOMEM = 2, /* workspace or probe buffer too small, host allocation failed */
    HEAT_ECUDA = 3,  /* CUDA runtime error, no usable sm_100 device */
    HEAT_ERANGE = 4  /* a property law is not strictly positive on the declared T range */
} heat_status;

/* Property law f(T).  The paper fits polynomials (23),(24) P:L245-248; BASELINE.json's
 * workloads use power laws.
 *   HEAT_LAW_CONST : f = c[0]
 *   HEAT_LAW_POWER : f = c[0] * (T / T_ref)^c[1]
 *   HEAT_LAW_POLY  : f = sum_{k=0..4} c[k] T^k   (ascending powers)                        */
enum { HEAT_LAW_CONST = 0, HEAT_LAW_POWER = 1, HEAT_LAW_POLY = 2 };
typedef struct {
    int32_t kind;
    int32_t reserved;
    double c[5];
    double T_ref;
} heat_law;

/* One material (the paper's index m, eq. (1)). */
typedef struct {
    heat_law k;         /* lambda_m(T), thermal conductivity                                 */
    heat_law cp;        /* c_Vm(T), specific heat                                            */
    double rho;         /* rho_m, density                                                    */
    int32_t is_heater;  /* X_m != 0 only in flagged layers (2) P:L70                         */
    int32_t reserved;
    heat_law src_shape; /* s(T): X = Q0 * s(T) * nu(t) * p^2(t); chi(T) of (25) P:L274 up to
                           a constant; CONST 1 for a temperature-independent source          */
} heat_layer;

/* Boundary condition of one side, (6) P:L90-95 generalised per side. */
enum { HEAT_BC_NEUMANN0 = 0, HEAT_BC_DIRICHLET = 1 };
typedef struct {
    int32_t kind;
    int32_t reserved;
    double value; /* Dirichlet temperature */
} heat_bc;

#define HEAT_MAX_LAYERS 16
#define HEAT_MAX_PROBES 64
#define HEAT_MAX_NR 8192 /* one thread block owns a whole z-line */

typedef struct {
    int32_t nr, nz, batch, nlayers;  /* nr,nz >= 3; batch >= 1; 1 <= nlayers <= HEAT_MAX_LAYERS */
    const double *r;                 /* host, nr, strictly ascending, r[0] >= 0 (9) P:L117      */
    const double *z;                 /* host, nz, strictly ascending                             */
    const heat_layer *layers;        /* host, nlayers                                            */
    const uint8_t *seg_layer;        /* host, batch*(nr-1): layer of radial segment (i,i+1).
                                        Node i is an interface node (rows (18)-(20) P:L176-192)
                                        iff its two segments differ; two interface nodes may
                                        not be adjacent                                          */
    heat_bc r_in, r_out, z_lo, z_hi; /* paper: N0,N0,N0,D(T0); BASELINE configs: N0,N0,D,D       */
    double T0;                       /* uniform initial temperature (5) P:L86 (if !T_init)       */
    const double *T_init;            /* optional [batch][nz][nr]; host unless T_init_is_device   */
    double dt;                       /* tau > 0                                                  */
    const double *Q0;                /* host, batch: source amplitude; NULL = no source          */
    int64_t steps_per_period;        /* t_prd / tau (4) P:L79; 0 = no source                     */
    int64_t steps_on;                /* t_src / tau; nu = 1 while (step in period) < steps_on    */
    int32_t transient_substeps;      /* (22) P:L212-217: the first tau of each period is taken as
                                        this many sub-steps of tau/substeps with
                                        p^2 = 1 - exp(-q/transient_k); paper: 100; 0 = Heaviside */
    int32_t face_mode;               /* lambda at a half node P:L127: 0 = lambda(mean T),
                                        1 = mean of lambda(T_a), lambda(T_b) (G3)      */
    double transient_k;              /* paper: 7                                                 */
    int32_t nprobes;                 /* <= HEAT_MAX_PROBES                                       */
    int32_t probe_every;             /* record after every probe_every-th step (>= 1 if nprobes) */
    const int32_t *probe_ij;         /* host, nprobes*(i,j)                                      */
    int32_t T_init_is_device;
    int32_t flags;                   /* HEAT_DESC_* bits, 0 = defaults                            */
    double T_lo, T_hi;               /* declared temperature range: every lambda_m, c_Vm must be
                                        strictly positive on it (HEAT_ERANGE otherwise; the
                                        paper's printed graphite c_V row is not, G11).
                                        T_hi <= T_lo disables the check                          */
    int32_t i_step, j_step;          /* stepped domain (reading G24 of "N_j" in
                                        the grid (9) P:L117 and of Fig. 1): the lines j > j_step end at
                                        node i_step (the core reaching the terminal) with zero flux (6) on
                                        the two new faces; the nodes i > i_step of those lines are not part
                                        of Omega: they are never solved, the line j_step + 1 of them mirrors
                                        line j_step (no flux through the step face), whatever T_init holds
                                        there.  0, 0 = rectangle.  2 <= i_step <= nr-2, 1 <= j_step <= nz-3;
                                        runs on the general line kernel                           */
} heat_desc;

/* heat_desc.flags: run this context on the general line kernel whatever the grid (needed by
 * heat_step_picard; also what HEAT_KERNEL=line in the environment does for every context). */
#define HEAT_DESC_GENERAL_KERNEL 1

/* Bytes of device workspace heat_create needs for this descriptor (0 if it is malformed). */
size_t heat_workspace_bytes(const heat_desc *d);

/* Right-hand side of the stability bound (21) P:L194-196,
 *   tau <= (min_j eta_j^2 / 2) * min_{m,T} rho_m c_Vm(T) / lambda_m(T),
 * the second minimum over the layers and T in [T_lo, T_hi] (1025 equidistant samples).
 * Host-only; does not touch the device. */
heat_status heat_stable_dt(const heat_desc *d, double T_lo, double T_hi, double *dt_limit);

/* Validate the descriptor, derive the per-node row tables, upload them into `workspace`
 * and initialise both field levels (initial condition (5), Dirichlet sides held from t=0).
 *   field_a, field_b : device, batch*nz*nr doubles each, 16-byte aligned, caller-owned
 *   workspace        : device, >= heat_workspace_bytes(d), 256-byte aligned, caller-owned
 *   probe_buf        : device, probe_cap doubles (may be NULL if nprobes == 0); records of
 *                      batch*nprobes doubles are appended until it is full, then dropped
 *   cuda_stream      : cudaStream_t used for the uploads; the call synchronises it
 * On failure *out is NULL and heat_last_error(NULL) describes why. */
heat_status heat_create(const heat_desc *d, void *field_a, void *field_b, void *workspace,
                        size_t workspace_bytes, void *probe_buf, size_t probe_cap,
                        void *cuda_stream, heat_ctx **out);

/* Enqueue n solver steps on cuda_stream (asynchronous).  A transient sub-step counts as one
 * step.  The schedule (tau_k, nu_k p_k^2) is derived from integer step counters only. */
heat_status heat_step(heat_ctx *c, int64_t n, void *cuda_stream);

/* Variant, not the paper's scheme: "for implicit difference schema with
 * coefficients depending on the sought-after function (temperature), one needs to make iterations for
 * evaluation of temperature at each time step", which the paper avoids by its switch-on
 * sub-stepping.  n solver steps, each as `iters` simple iterations on the coefficients
 * (reading G23): T^(0) = T; T^(s+1) solves (8)-(20) with every lambda_m, c_Vm and X_m
 * evaluated at T^(s), the current level T staying in rho c_V (T^ - T)/tau and in Lambda_j[T];
 * T^ = T^(iters).  iters = 1 is heat_step.  One kernel launch per iteration.
 *   field_c : device, batch*nz*nr doubles, 16-byte aligned, caller-owned: the second iterate buffer.
 *             It is scratch between calls (never the current level); its z-boundary lines are set
 *             up on the first call with this pointer and after heat_set_field / heat_set_line.
 * Needs a context created with HEAT_DESC_GENERAL_KERNEL (HEAT_EINVAL otherwise).  Schedule, step
 * counter and probe records advance per solver step, as in heat_step. */
heat_status heat_step_picard(heat_ctx *c, int64_t n, int32_t iters, void *field_c, void *cuda_stream);

/* Copy the current level of batch member b ([nz][nr], r fastest) to dst.  Asynchronous if
 * dst is a device pointer; synchronises the stream if dst is host memory. */
heat_status heat_get_field(heat_ctx *c, int32_t b, double *dst, int32_t dst_is_device,
                           void *cuda_stream);

/* Overwrite the current level of batch member b (both levels' z-boundary lines included)
 * and set the solver step counter (checkpoint / resume, snapshot-seeded parity windows). */
heat_status heat_set_field(heat_ctx *c, int32_t b, const double *src, int32_t src_is_device,
                           int64_t step_index, void *cuda_stream);

/* One z-line (nr doubles, r fastest) of the current level of batch member b: read it, or overwrite it
 * in both levels.  These are what a z-slab multi-GPU run exchanges after every step (SURVEY 8(e):
 * P:L125 couples line j only to lines j -+ 1 of the old level): a slab's halo line is a Dirichlet z
 * line, which no step ever writes (G17), refreshed with the neighbour's edge line.  Asynchronous on
 * cuda_stream for device pointers; a host pointer synchronises the stream. */
heat_status heat_get_line(heat_ctx *c, int32_t b, int32_t j, double *dst, int32_t dst_is_device, void *cuda_stream);
heat_status heat_set_line(heat_ctx *c, int32_t b, int32_t j, const double *src, int32_t src_is_device, void *cuda_stream);

/* z-slab multi-GPU run with direct peer stores instead of heat_get_line / heat_set_line:
 * tell this context where a neighbour slab keeps its two field levels.  From then on every heat_step
 * also stores this slab's first interior line (side 0: the neighbour below) or last interior line
 * (side 1: the neighbour above) of the NEW level into the neighbour's halo line -- its last line
 * (side 0) or its line 0 (side 1) -- of the neighbour's NEXT level: the level buffer with the same
 * position (a / b) as this context's next level.  The store is issued by the step kernel itself (a TMA
 * store in the tband kernel, plain stores in the line kernel), so over NVLink the exchange overlaps the
 * rest of the step; no other call moves halo data.
 *   peer_field_a, peer_field_b : the field_a, field_b the neighbour passed to ITS heat_create, as
 *                                addresses valid on this device (same GPU, or peer-mapped: P2P access
 *                                enabled / cudaIpcOpenMemHandle); NULL, NULL switches the side off
 *   peer_nz                    : the neighbour's nz (its halo lines included); nr and batch are this context's
 * Contract: all slabs start from the same level (a freshly created context, or the same number of steps)
 * and advance in lock step -- one heat_step(1) each, then a synchronisation between the ranks (the
 * neighbour reads the stored line in its next step) -- so the level written is never the one a
 * neighbour's running step reads.  The side that faces a neighbour must be a Dirichlet z line.
 * Available for contexts on the tband and the line kernel (HEAT_EINVAL otherwise); multi-step
 * persistent launches are off while a peer is set, and heat_step_picard with iters > 1 is refused (its
 * iterates would need an exchange per iteration). */
heat_status heat_set_halo_peer(heat_ctx *c, int32_t side, void *peer_field_a, void *peer_field_b, int32_t peer_nz);

/* Drain the probe trace: synchronise cuda_stream, copy up to max doubles (whole records of
 * batch*nprobes doubles, order [record][batch][probe]) to dst_host, and rewind the device
 * buffer.  *n_written = doubles copied; *n_dropped (optional) = records lost to overflow. */
heat_status heat_probe(heat_ctx *c, double *dst_host, int64_t max, int64_t *n_written,
                       int64_t *n_dropped, void *cuda_stream);

/* (tau_k, amplitude_k) of solver step s under this context's schedule (host-only). */
heat_status heat_schedule(const heat_ctx *c, int64_t s, double *tau, double *amp);

/* Solver steps enqueued so far. */
int64_t heat_step_index(const heat_ctx *c);

/* Number of kernels this context has launched since creation (bench accounting). */
int64_t heat_launch_count(const heat_ctx *c);

/* Name of the kernel variant heat_step launches for this context, e.g. "line<M=16,G=512>". */
const char *heat_kernel_name(const heat_ctx *c);

/* Message of the last failure on this context (c != NULL) or of the last failed
 * heat_create / heat_stable_dt on the calling thread (c == NULL).  Never NULL. */
const char *heat_last_error(const heat_ctx *c);

void heat_destroy(heat_ctx *c);

/* ---- bench accounting (HEAT_BENCH): not part of the method ------------------------------------
 * heat_launch_count and heat_kernel_name above belong here as well: they exist so that bench.py
 * can report `gpu_launches` and name the kernel its roofline line is about.
 *
 * Measured-peak helper for the ALU co-limit of the roofline: runs a dependent-chain-free DFMA loop on
 * every SM and returns the achieved fp64 FMA rate in TFLOP/s (2 flops per FMA); iters per thread.
 *   scratch, scratch_bytes : caller-owned device buffer, >= heat_fp64_peak_scratch_bytes() bytes
 *                            (like every other call, the library allocates no device memory)
 * Synchronises cuda_stream. */
size_t heat_fp64_peak_scratch_bytes(void);
heat_status heat_fp64_peak(int64_t iters, void *scratch, size_t scratch_bytes, void *cuda_stream, double *tflops);

/* ---- allocation-free set-up ---------------------------------------------------------------------
 * heat_create for callers that cannot call cudaMalloc (set-up next to CUDA graph capture, serving loops,
 * harnesses that forbid it): the same call without the workspace arguments.  The row tables that every
 * step kernel reads (the coefficients of rows (13), (15), (18) P:L140-192, the z factors
 * of (11) P:L125, the law tables) live in a static device array of HEAT_STATIC_WORKSPACE_BYTES inside
 * the library, which every GPU that loads the library holds until the process exits.  The call
 * allocates no device memory (neither does any other call of this library: they take caller-owned
 * buffers); field_a, field_b, probe_buf are the caller's as in heat_create.
 *   - HEAT_ENOMEM with a message naming both sizes if heat_workspace_bytes(d) exceeds the array;
 *     the five BASELINE.json configurations need 0.01 - 2.7 MiB (configs[3]: 2 772 992 B).
 *   - The array is shared by every heat_create_static context of the process on that device and keeps
 *     the previous one's contents; each call clears the part it uses before the upload.  Hence at most
 *     ONE live heat_create_static context per device: creating a second one overwrites the tables
 *     under the first, and calls that overlap on the GPU (a step of the first context still running
 *     on another stream while the second is created) race.  Destroy the context, and let its work
 *     finish, before the next heat_create_static on the same device.
 * Everything else (heat_step, heat_get_field, heat_probe, heat_destroy ...) is used as with heat_create,
 * and the results are bitwise those of heat_create (tests/test_zz_no_alloc.py). */
#define HEAT_STATIC_WORKSPACE_BYTES (4u << 20)
size_t heat_static_workspace_bytes(void);
heat_status heat_create_static(const heat_desc *d, void *field_a, void *field_b, void *probe_buf,
                               size_t probe_cap, void *cuda_stream, heat_ctx **out);

#ifdef __cplusplus
}
#endif
#endif /* HEAT_B200_H */
