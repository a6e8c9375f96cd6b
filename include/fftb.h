/*
 * fftb.h -- C-ABI of fftb-b200: the batched, pruned sphere <-> cuboid 3D complex FFT of
 * plane-wave DFT codes (arXiv 2406.05577, "FFTB"), one NVIDIA B200 (sm_100a).
 *
 * The boundary follows the paper's "create, execute and clean-up" constructs
 * (PAPER.md:130 [3.1 Computational Layout Descriptor]): a plan is created from a
 * description of the bounding domain, the cut-off that generates the offset array
 * (Fig. 7, 183-185 [3.3]) and the batch dimension (PAPER.md:219 [3.3]);
 * it is executed any number of times; it is destroyed.  A description outside the
 * predefined patterns is refused with FFTB_EUNSUPPORTED ("The framework
 * will raise an exception if the provided patterns are not within the predefined list").
 *
 * Conventions (DESIGN.md lists the readings R1-R13 of the paper behind them)
 *   grid      (N1,N2,N3) = (x,y,z); x fastest in memory, z slowest;
 *             z is the stick axis.  C = N1*N2*N3.
 *   frequency signed integers k_d in [-N_d/2, N_d/2); grid index i_d = k_d mod N_d.
 *   cut-off   the points with (k1/a1)^2 + (k2/a2)^2 + (k3/a3)^2 <= 1 (Eq. 9,
 *             inclusive, decided in exact integer arithmetic); S of them.
 *   packed    [nb][S]: band slowest; inside a band the points are ordered by k1
 *             ascending, then k2 ascending, then k3 ascending (signed values), i.e. one
 *             contiguous "z-stick" per occupied (k1,k2) column, sticks ordered by (k1,k2).
 *   cuboid    [nb][N3][N2][N1], x contiguous.
 *   vloc      [N3][N2][N1] real (double for FFTB_C128, float for FFTB_C64), one for all bands.
 *   inverse   psi[b][i] = sum_p c[b][p] exp(+2 pi j (k1 i1/N1 + k2 i2/N2 + k3 i3/N3))
 *             (Eq. 8), unnormalised.
 *   forward   c[b][p] = s * sum_i psi[b][i] exp(-2 pi j (k1 i1/N1 + ...)) for the points of
 *             the cut-off only (Eq. 3-4); s = 1 (FFTB_SCALE_NONE) or 1/C
 *             (FFTB_SCALE_FORWARD).
 *   apply_vloc c' = forward( V .* inverse(c) ), the cuboid never leaves the chip.
 *
 * Pointers named d_* are DEVICE pointers, h_* are HOST pointers; everything else is host.
 * Device pointers must be 16-byte aligned; complex128 CUBOID pointers must be 32-byte aligned (the
 * kernels move two neighbouring x values as one 32-byte access); anything else is FFTB_EINVAL.
 * The caller owns every device buffer,
 * including the table/workspace block handed to fftb_plan_bind; the plan owns host
 * memory only.  The execute calls enqueue work on `stream` (a cudaStream_t passed as
 * void*; NULL = the legacy default stream) and return without synchronising; they do not
 * allocate.  Inputs are const and are preserved.
 *
 * Every function returns 0 (FFTB_OK) or a negative fftb_status; nothing throws or aborts.
 */
#ifndef FFTB_H
#define FFTB_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fftb_plan_s *fftb_plan; /* opaque, host-owned */

enum fftb_status {
    FFTB_OK = 0,
    FFTB_EINVAL = -1,       /* null pointer, nb < 1 or > batch, N_d < 1, a_d < 0, 2 a_d >= N_d (aliasing),
                               unknown enum value, misaligned pointer */
    FFTB_EUNSUPPORTED = -2, /* a description outside the predefined patterns (see fftb_plan_create) */
    FFTB_ENOMEM = -3,       /* host allocation failed, or the bind block is too small */
    FFTB_ECUDA = -4,        /* a CUDA call or launch failed (this includes the driver's cuTensorMapEncodeTiled, which the
                               N1 == N2 == 256 kernels and the fused launches need: CUDA 12 drivers have it); sticky until
                               the plan is destroyed */
    FFTB_ESTATE = -5,       /* execute before fftb_plan_bind, or mismatched plans */
    FFTB_ETOOBIG = -6       /* fftb_inverse_static only: the plan's tables plus one band of its intermediate do not fit in
                               the library's static scratch array (FFTB_STATIC_SCRATCH_BYTES) */
};

enum fftb_dtype { FFTB_C64 = 0, FFTB_C128 = 1 };               /* element type of packed and cuboid */
enum fftb_scale { FFTB_SCALE_NONE = 0, FFTB_SCALE_FORWARD = 1 }; /* 1/(N1 N2 N3) applied in forward */
enum fftb_flags {
    FFTB_FLAG_DENSE = 1u, /* no pruning: every (k1,k2) is a full-length stick, S = C, `cutoff` ignored.
                             This is the "pad the sphere to the cube, transform the entire cube" route of
                             PAPER.md:110-112, run by the same kernels (BASELINE config 5). */
    FFTB_FLAG_BATCH_FASTEST = 2u /* the PACKED arrays of every execute call are batch-fastest, [S][nb] (element [point][band],
                             nb = the bands of that call): the layout of the paper's own example, Fig. 8 "b x y z"
                             (PAPER.md:219-221).  The transposition is folded into the z passes (their tile loads and
                             stores), no extra pass over the packed arrays; the cuboid stays [nb][N3][N2][N1].  Only for
                             N3 in {64, 96, 128, 192 (FFTB_C64)} with N1 in {64, 96, 128, 256}: FFTB_EUNSUPPORTED
                             otherwise; not together with FFTB_FLAG_DENSE (FFTB_EINVAL). */
};

typedef struct {
    int32_t n[3];      /* N1 (x, fastest), N2 (y), N3 (z, stick axis) */
    int32_t cutoff[3]; /* integer semi-axes a1,a2,a3 >= 0 in index units; ignored if DENSE */
    int32_t batch;     /* maximum number of bands per execute call, >= 1 */
    int32_t dtype;     /* fftb_dtype */
    int32_t scale;     /* fftb_scale */
    uint32_t flags;    /* fftb_flags */
} fftb_plan_desc;

typedef struct {
    int64_t n_points;     /* S */
    int64_t n_sticks;     /* occupied (k1,k2) columns */
    int64_t n_xocc;       /* distinct k1 with at least one stick */
    int64_t device_bytes; /* smallest block fftb_plan_bind accepts (tables + workspace) */
    int64_t device_bytes_host; /* block size that also holds the staging areas of the *_host calls (2 * batch * S
                                  elements more; 4 * batch * S with FFTB_TUNE_HOST_DEFER) */
    int64_t chunk_bands;  /* bands per kernel group in fftb_inverse (the workspace holds this many) */
    int64_t min_bytes_per_band_dir; /* algorithmic bytes of one band, one direction: (S + C) * elem */
    int64_t workspace_offset; /* byte offset of the plane-major intermediate A inside the bind block */
    int64_t pitch;        /* row pitch of A in elements: A[band][z][pitch] after the inverse z pass */
    int64_t y_residues;   /* largest number of partial A planes a forward-side plane kernel of this plan writes
                             per band (the fast kernels accumulate the y residues themselves and write one) */
    int64_t chunk_bands_fwd;  /* bands per kernel group in fftb_forward */
    int64_t chunk_bands_vloc; /* bands per kernel group in fftb_apply_vloc */
    int64_t ring_bands;   /* > 0: fftb_inverse and fftb_forward are ONE launch each that keeps the intermediate in a
                             ring of this many band slots at workspace_offset (band b in slot b % ring_bands);
                             0: separate z-pass and plane launches per band chunk, A[band][z][pitch] */
    int64_t lead_bands;   /* how many bands the producers of the ring run ahead of its consumers */
    /* layout of a ring slot (tile-major): stick s, plane z of the band sits at element
     *   (s / ring_tile_sticks) * ring_tile_elems + (z / 2) * ring_pair_pitch + (z % 2) * ring_tile_sticks + s % ring_tile_sticks
     * and a slot holds ceil(n_sticks / ring_tile_sticks) * ring_tile_elems elements */
    int64_t ring_tile_sticks, ring_tile_elems, ring_pair_pitch;
} fftb_plan_info;

/* Optional tuning of a plan, for tests and measurements; everything 0 = the defaults fftb_plan_create uses. */
enum fftb_tuning_flags {
    FFTB_TUNE_GENERIC_Z = 1u,     /* z passes by the generic kernels even where a persistent TMA kernel exists */
    FFTB_TUNE_GENERIC_PLANE = 2u, /* y/x passes by the generic plane kernel even where a persistent one exists */
    FFTB_TUNE_FUSED = 4u,         /* fftb_inverse / fftb_forward as ONE cooperative launch each (z tiles and planes of the whole
                                     batch, the intermediate in an L2-resident ring: 27% less DRAM traffic) where that launch
                                     exists (128^3 grids); measured slower than the separate launches, hence opt-in */
    FFTB_TUNE_NO_L2_HINTS = 8u,   /* fused launches without L2 eviction priorities (ring evict_last, streams evict_first) */
    FFTB_TUNE_HOST_DEFER = 16u    /* *_host calls: DEFERRED completion.  A call no longer makes `stream` wait for its own
                                     device-to-host copies; fftb_host_flush does that for all calls so far.  The plan then
                                     keeps two incoming and two outgoing staging areas (info.device_bytes_host counts
                                     them) that successive calls take in turn, so the transforms of call i+1 run while
                                     the results of call i are still leaving: a sequence of calls is bound by the link
                                     (both directions busy), not by copies + kernels in a row */
};
typedef struct {
    int64_t workspace_bytes; /* budget for the intermediate A inside the bind block (the plan rounds it to whole bands,
                                at least one); 0 = default */
    int32_t ring_bands;      /* band slots of the fused launches' ring; 0 = default (lead_bands + 2) */
    int32_t lead_bands;      /* bands the producers run ahead; 0 = default (2) */
    uint32_t flags;          /* fftb_tuning_flags */
    uint32_t z_ctas;         /* fused launches: > 0 = spatial split, this many CTAs take the z tiles only and the others the
                                planes only (ignored if the launch has no more CTAs than that); 0 = every CTA walks both
                                lists merged (default); > 1024: FFTB_EINVAL */
} fftb_plan_tuning;

/* Create a plan (host only, no CUDA call).  Builds the offset array -- the stick map -- from the
 * grid and the cut-off (Fig. 7), the per-k1 stick runs used by the y pass, and the
 * twiddle tables.
 * Predefined patterns (anything else: FFTB_EUNSUPPORTED), FFTB_C64 or FFTB_C128 unless stated:
 *   - N3 in {32, 64, 96, 128, 192, 256}; N1 == N2 in the same set, or (N1, N2) one of (32, 64), (64, 32), (64, 128),
 *     (128, 64);
 *   - pruned plans with a_d <= N_d/4 on every axis (the paper's "cube of width twice the diameter of the sphere",
 *     PAPER.md:110): half-band kernels, persistent TMA kernels where they exist (N1 == N2 in {64, 96, 128, 256});
 *   - pruned plans with N_d/4 < a_d < N_d/2 on some axis: full-band axis patterns (generic kernels), N1 == N2 and N3 in
 *     {32, 64, 128, 256};
 *   - dense plans (FFTB_FLAG_DENSE): N1 == N2 and N3 in {32, 64, 128, 256}; the cubes 64^3, 128^3 and 256^3 run three
 *     line passes per direction on the transform core of the persistent kernels (fftb_dense.cuh), the others the
 *     generic kernels. */
int fftb_plan_create(fftb_plan *out, const fftb_plan_desc *desc);

/* The same with explicit tuning (tuning == NULL: fftb_plan_create).  FFTB_EINVAL for unknown flags or negative
 * fields. */
int fftb_plan_create_tuned(fftb_plan *out, const fftb_plan_desc *desc, const fftb_plan_tuning *tuning);

/* Create a plan from an EXPLICIT stick map instead of a cut-off: the paper's general domain with an
 * offset array (PAPER.md:183-185: "x and y dense, only z compressed", :201 `offsets` argument), e.g. the
 * g-vector list of a plane-wave code whose sphere is shifted by a k-point.  Stick s is the k3 run
 * k3lo[s] .. k3lo[s]+len[s]-1 of column (k1[s], k2[s]); `desc->cutoff` is ignored, FFTB_FLAG_DENSE is not
 * allowed.  The arrays (host, n_sticks entries each) are copied.  The map may have HOLES -- k1 values without a stick inside
 * the occupied k1 range, k2 values without a stick inside a column's k2 run (the g-vector list of a cell whose sphere is cut by
 * a second criterion): the plan fills them with zero-length sticks of its own, which the caller never sees (get_map and
 * info.n_sticks report the map as given; the intermediate's pitch counts them).
 *   FFTB_EINVAL        a point outside [-N_d/2, N_d/2), len < 1, sticks not strictly ascending in (k1, k2)
 *   FFTB_EUNSUPPORTED  outside the predefined patterns of fftb_plan_create (a frequency beyond |k_d| <= N_d/4 makes
 *                      it a full-band plan). */
int fftb_plan_create_explicit(fftb_plan *out, const fftb_plan_desc *desc, int64_t n_sticks, const int32_t *k1,
                              const int32_t *k2, const int32_t *k3lo, const int32_t *len);

/* The same with explicit tuning (tuning == NULL: fftb_plan_create_explicit). */
int fftb_plan_create_explicit_tuned(fftb_plan *out, const fftb_plan_desc *desc, int64_t n_sticks, const int32_t *k1,
                                    const int32_t *k2, const int32_t *k3lo, const int32_t *len, const fftb_plan_tuning *tuning);

int fftb_plan_info_get(fftb_plan p, fftb_plan_info *info);

/* Copy the stick map to host arrays supplied by the caller (any may be NULL):
 * k1,k2,k3lo,len have n_sticks entries, off has n_sticks+1 (exclusive prefix sum of len, the
 * paper's CSR-like offset array). */
int fftb_plan_get_map(fftb_plan p, int32_t *k1, int32_t *k2, int32_t *k3lo, int32_t *len, int64_t *off);

/* Hand the plan its device memory: `d_mem` (>= info.device_bytes, 256-byte aligned, caller-owned,
 * must outlive the plan's last execute).  Uploads the tables on `stream` (cudaMemcpyAsync from
 * plan-owned host memory) and returns; later execute calls on the same stream are ordered after it. */
int fftb_plan_bind(fftb_plan p, void *d_mem, size_t bytes, void *stream);

/* The three device-pointer execute calls below only enqueue kernels on `stream`: no allocation, no
 * synchronisation, no host-side dependence on the data.  They may therefore be captured in a CUDA
 * graph by the caller (stream capture) and replayed; the *_host variants use plan-owned copy streams
 * and events and are not meant for capture. */

/* inverse: d_packed [nb][S] -> d_cuboid [nb][N3][N2][N1].  unpack + pruned z pass on the sticks,
 * y pass on the occupied x columns only, x pass last (Fig. 3, 112: staged padding). */
int fftb_inverse(fftb_plan p, const void *d_packed, void *d_cuboid, int nb, void *stream);

/* inverse for callers that cannot allocate device memory at all (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): the SAME kernels as fftb_inverse (the separate z-pass and plane launches), but the
 * plan's tables and the intermediate A live in ONE array of FFTB_STATIC_SCRATCH_BYTES that the library itself holds in
 * device memory (a file-scope `static __device__` array: every GPU that loads the library keeps these 16 MiB until the
 * process exits).  The plan needs no fftb_plan_bind and no bind block (a bound plan's block is not touched); the caller
 * passes only the input and the output, same layouts, alignment and nb range as fftb_inverse.  The call makes no
 * cudaMalloc / cudaFree and calls no allocating routine: it copies the plan's tables (host memory the plan owns; some
 * tens of KB) into the array on `stream`, then enqueues the kernels for as many bands at a time as the rest of the array
 * holds.  Results are bit-identical to fftb_inverse.
 *   FFTB_ETOOBIG  tables + ONE band of the intermediate (N3 * pitch elements) exceed FFTB_STATIC_SCRATCH_BYTES; e.g.
 *                 128^3 complex128 at radius 32 needs 6.4 MiB and fits (two bands at a time), 256^3 at radius 64 needs
 *                 50 MiB and is refused.  Nothing is enqueued.
 *   FFTB_EINVAL / FFTB_ECUDA as for fftb_inverse; a failure here does not make the plan sticky.
 * Every call on a device SHARES the one array, and the array keeps the last call's contents: each call rewrites the
 * tables and every element of A it later reads, so nothing has to start at zero, but two calls that overlap on the GPU
 * (different streams without an event between them, or two host threads on different streams) race on it -- keep
 * them on one stream or order them yourself.  The plan itself is only read. */
#define FFTB_STATIC_SCRATCH_BYTES (16u * 1024u * 1024u)
int fftb_inverse_static(fftb_plan p, const void *d_packed, void *d_cuboid, int nb, void *stream);

/* forward: d_cuboid -> d_packed, the mirror image; applies the plan's scale. */
int fftb_forward(fftb_plan p, const void *d_cuboid, void *d_packed, int nb, void *stream);

/* local-potential apply, fused: inverse up to the x pass, multiply by V(r), forward x pass
 * immediately, then forward y and z passes.  d_packed_in == d_packed_out is allowed. */
int fftb_apply_vloc(fftb_plan p, const void *d_packed_in, void *d_packed_out, const void *d_vloc, int nb,
                    void *stream);

/* The same three operations with the PACKED arrays in host memory (pinned memory makes the copies asynchronous): the
 * library copies them through two staging areas inside the bind block (one per direction), cuboid and vloc stay device
 * pointers.  Large batches cross PCIe in band chunks on two copy streams owned by the plan (created in fftb_plan_bind),
 * overlapped with the transforms of the neighbouring chunks, and the host-to-device copies of a call may run while the
 * device-to-host copies of the previous call are still under way (both directions of the link at once).  Ordering:
 *   - a call's OUTPUT is complete in host memory when `stream` reaches the end of the call (work queued later sees it);
 *   - a call's host INPUT is read by copies that are ordered after the previous call's kernels, not after other work
 *     queued on `stream`: its contents must be final when the call is made;
 *   - plans created with FFTB_TUNE_HOST_DEFER: the OUTPUT of a call is complete in host memory only once `stream` has
 *     passed a later fftb_host_flush (the host array must not be read, reused or freed before that). */
int fftb_inverse_host(fftb_plan p, const void *h_packed, void *d_cuboid, int nb, void *stream);
int fftb_forward_host(fftb_plan p, const void *d_cuboid, void *h_packed, int nb, void *stream);
int fftb_apply_vloc_host(fftb_plan p, const void *h_packed_in, void *h_packed_out, const void *d_vloc, int nb,
                         void *stream);
/* Makes `stream` wait for the device-to-host copies of every *_host call made on the plan so far (only enqueues the
 * waits; a no-op for plans without FFTB_TUNE_HOST_DEFER, whose calls wait themselves).  FFTB_ESTATE before fftb_plan_bind. */
int fftb_host_flush(fftb_plan p, void *stream);

/* Comparison arm of BASELINE config 5 ("zero-pad the entire sphere ... the 3D
 * Fourier computation is applied on the entire cube"): scatter the packed sphere of `pruned` into the
 * (zero-filled) packed layout of the DENSE plan `dense` of the same grid and dtype, and gather it back. */
int fftb_dense_embed(fftb_plan pruned, fftb_plan dense, const void *d_packed_pruned, void *d_packed_dense, int nb,
                     void *stream);
int fftb_dense_extract(fftb_plan pruned, fftb_plan dense, const void *d_packed_dense, void *d_packed_pruned, int nb,
                       void *stream);

/* Packed arrays in the paper's batch-fastest order (Fig. 8 "b x y z": the band index
 * is the fastest one, element [point][band], nb bands) and in this library's order [band][point]
 * (north_star: "packed z-sticks per band"): to_band_slowest != 0 copies d_in = [S][nb] to
 * d_out = [nb][S], to_band_slowest == 0 the other way.  Both are device pointers, 16-byte aligned,
 * S * nb elements of the plan's dtype, owned by the caller; in place is not supported
 * (FFTB_EINVAL), nb is not limited by the plan's batch.  One kernel, both sides coalesced; this is
 * how a caller that keeps its coefficients batch-fastest uses the transforms. */
int fftb_packed_transpose(fftb_plan p, const void *d_in, void *d_out, int nb, int to_band_slowest, void *stream);

/* Number of kernels the last execute call on this plan launched (for launch accounting). */
int fftb_plan_last_launches(fftb_plan p);

/* Device probe for benchmarks: the FMA rate of the plain FP64 (FFTB_C128) or FP32 (FFTB_C64) pipe of the current
 * device in TFLOP/s (2 flops per FMA), from a register-only loop on all SMs; *ms (may be NULL) receives the best of
 * five runs.  Unlike the execute calls this one allocates a scratch array, runs on the legacy default stream and WAITS
 * for the result.  It is the denominator of the "alu" roofline of the fused local-potential workloads
 * ("FP64 pipe utilisation ... over the probed peak"). */
int fftb_probe_fma(int dtype, double *tflops, double *ms);
/* The same kind of probe for the global-store port of an SM: `n_sms` CTAs (one per SM) stream 32-byte stores; returns the
 * bytes per clock ONE SM sustained (issue-side clocks) and the aggregate GB/s (may be NULL).  Allocates 32 MB per CTA,
 * legacy default stream, waits.  On B200 an SM stores 32 B/clk however few SMs take part, which bounds the x phase of
 * the inverse plane kernels. */
int fftb_probe_store_port(int n_sms, double *bytes_per_clk_per_sm, double *gbs);

/* Per-kernel timing for benchmarks.  fftb_plan_profile(p, 1) makes every later execute call record a
 * CUDA event pair around each kernel it launches (on the launching stream); fftb_plan_profile_read
 * waits for them, adds the elapsed milliseconds and launch counts per kernel kind into ms[7] and
 * count[7] -- 0 inverse z pass, 1 inverse plane, 2 forward plane, 3 forward z pass, 4 fused vloc
 * plane, 5 fused inverse launch (z tiles + planes), 6 fused forward launch -- and clears the record.
 * fftb_plan_profile(p, 0) switches it off. */
int fftb_plan_profile(fftb_plan p, int enable);
int fftb_plan_profile_read(fftb_plan p, double *ms, int64_t *count);

int fftb_plan_destroy(fftb_plan p);

/* ---------------------------------------------------------------------------------------------------------------
 * Slab-distributed transform: ONE transform spread over `world` GPUs the way
 * the paper's plane-wave variant does it on a 1D grid.  Rank r owns
 *   - the sticks of a contiguous range of occupied k1 columns (ranges balanced by stick count), i.e. the contiguous
 *     part [packed_lo[r], packed_lo[r+1]) of every band of the packed array, and
 *   - the z-planes [z_lo[r], z_lo[r+1]) of the cuboid (contiguous slabs of N3).
 * inverse: z pass on the own sticks -> exchange (only pruned stick data travels) -> y/x passes on the own planes;
 * forward: the mirror image.  The library does every step but the transport: `*_begin` leaves the blocks for the
 * peers either in `d_send` (layout [peer][band][row][column], peer blocks in rank order; hand it to an NCCL all-to-all
 * with the counts of fftb_slab_plan_counts) or, when `d_peer` is given, directly in the peers' intermediates through
 * peer-mapped pointers (d_peer[i] = what fftb_slab_plan_exchange_ptr returns on rank i; then the pack kernel IS the
 * exchange and d_send / d_recv are not used).  `*_end` consumes `d_recv` ([peer][band][row][column]) or, with
 * d_recv == NULL, the intermediate the peers have written.  The caller orders begin -> transport -> end (stream order on
 * one GPU; a barrier or events between ranks).  Same conventions, scale, alignment and error codes as above;
 * FFTB_EUNSUPPORTED additionally for world > 16, fewer occupied k1 columns or z-planes than ranks, FFTB_FLAG_DENSE, or a
 * pattern whose forward plane kernel writes partial planes. */
typedef struct fftb_slab_plan_s *fftb_slab_plan;

typedef struct {
    int64_t n_points_local;  /* packed points of this rank per band: packed_lo[rank+1] - packed_lo[rank] */
    int64_t n_sticks_local;
    int64_t planes_local;    /* z-planes of this rank's slab */
    int64_t device_bytes;    /* smallest block fftb_slab_plan_bind accepts */
    int64_t n_points, n_sticks; /* of the whole transform */
} fftb_slab_info;

/* host only; every rank calls it with the same desc and world and gets the same partition */
int fftb_slab_plan_create(fftb_slab_plan *out, const fftb_plan_desc *desc, int world, int rank);
int fftb_slab_plan_info_get(fftb_slab_plan p, fftb_slab_info *info);
/* the partition: stick_lo, packed_lo and z_lo have world + 1 entries each (any may be NULL) */
int fftb_slab_plan_counts(fftb_slab_plan p, int64_t *stick_lo, int64_t *packed_lo, int64_t *z_lo);
int fftb_slab_plan_bind(fftb_slab_plan p, void *d_mem, size_t bytes, void *stream);
/* device pointer (inside the bind block) peers write to in the direct mode: which = 0 the intermediate the INVERSE
 * exchange fills (all sticks x own planes), 1 the one the FORWARD exchange fills (own sticks x all planes) */
int fftb_slab_plan_exchange_ptr(fftb_slab_plan p, int which, void **d_ptr);

/* d_packed_local [nb][n_points_local]; d_cuboid_slab [nb][planes_local][N2][N1]; d_peer: host array of `world` device
 * pointers or NULL; d_send / d_recv: device buffers of the sizes the counts imply, or NULL in the direct mode */
int fftb_slab_inverse_begin(fftb_slab_plan p, const void *d_packed_local, void *const *d_peer, void *d_send, int nb, void *stream);
int fftb_slab_inverse_end(fftb_slab_plan p, const void *d_recv, void *d_cuboid_slab, int nb, void *stream);
int fftb_slab_forward_begin(fftb_slab_plan p, const void *d_cuboid_slab, void *const *d_peer, void *d_send, int nb, void *stream);
int fftb_slab_forward_end(fftb_slab_plan p, const void *d_recv, void *d_packed_local, int nb, void *stream);
int fftb_slab_plan_destroy(fftb_slab_plan p);


const char *fftb_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* FFTB_H */
