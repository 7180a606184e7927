/* elg.h -- C ABI of libelg: B200-native (sm_100a) tracking of a 6-D fp64 macroparticle bunch through a
 * lumped-element beamline -- the data-parallel hot path of arXiv:1710.07350 ("GPU acceleration and
 * performance of the particle-beam-dynamics code Elegant").
 *
 * Citations: "PAPER.md:NN" = line of the paper text; "Gk" = reading k in DESIGN.md ("Readings").
 *
 * Problem statement: a bunch of particles traverses a succession of elements.  Per-particle
 * element maps (first- to third-order transport maps), particle loss
 * (PAPER.md:139-141), longitudinal and transverse wakes built from a histogram and an array convolution
 * and beam-moment reductions are all computed by CUDA kernels
 * of this library; nothing is computed on the host and there is no
 * CPU fallback: every compute call fails with ELG_ECUDA when no device is usable.
 *
 * Conventions
 *  - Every call returns an int32 status: ELG_OK = 0, negative = error.  No exceptions or aborts cross the
 *    ABI; elg_last_error() returns a thread-local message for the last failing call.
 *  - "d_" arguments are DEVICE pointers, "h_" arguments are HOST pointers.  The library allocates no
 *    device memory: the caller (PyTorch in this repo) allocates the particle store and one workspace and
 *    lends them to the bunch handle for its lifetime.  While a bunch handle exists the caller must not
 *    write those buffers (the paper nulls the host pointer while the device owns the data).
 *  - Calls are asynchronous on the stream given to elg_bunch_create, except those that return host data
 *    (elg_moments, elg_lost, elg_n_alive, elg_bunch_read, and elg_track when it has host outputs), which
 *    synchronise that stream (the paper's finishReductionStreams moment).
 *  - Coordinates (G1): 0 x [m], 1 x' [rad], 2 y [m], 3 y' [rad], 4 s [m] (total path length,
 *    PAPER.md:75-77), 5 delta = (p-p0)/p0; plus an int64 particle ID.
 *
 * Particle store layout (struct of arrays): seven arrays, each elg_soa_stride(n0)
 * elements of 8 bytes apart, in the order x, x', y, y', s, delta (fp64) and ID (int64); the buffer is
 * 7 * stride * 8 bytes and must be 256-byte aligned.  The live particles are the prefix [0, n_alive) of
 * every array, in their original relative order (stable compaction, G18/G19).
 */
#ifndef ELG_H
#define ELG_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { ELG_OK = 0, ELG_EINVAL = -1, ELG_ENOMEM = -2, ELG_ECUDA = -3, ELG_ESTATE = -4, ELG_ECAPACITY = -5 };

/* element types (glossary PAPER.md:175; Table I rows PAPER.md:143-165) */
enum { ELG_DRIFT = 1, ELG_MATRIX = 2, ELG_RFKICK = 3, ELG_RCOL = 4, ELG_ECOL = 5, ELG_WAKE = 6, ELG_HISTO = 7,
       ELG_MATRIX2 = 8, ELG_TRWAKE = 9, ELG_MATRIX3 = 10 };
/* histogram window modes (G10) */
enum { ELG_WIN_EXPLICIT = 0, ELG_WIN_AUTO_MINMAX = 1, ELG_WIN_AUTO_TABLE = 2 };
/* wake kinds (G12) */
enum { ELG_WAKE_RESONATOR = 0, ELG_WAKE_TABLE = 1, ELG_WAKE_RESONATOR_T = 2 /* transverse resonator, TRWAKE only */,
       ELG_WAKE_RESONATOR_REC = 3 /* the resonator of kind 0 evaluated by the O(nb) recurrence (G37), WAKE only */ };
/* when elg_track records moments (G26) */
enum { ELG_MOM_NONE = 0, ELG_MOM_TURN = 1, ELG_MOM_ELEMENT = 2 };

/* One beamline element; all pointers are HOST pointers, copied by elg_beamline_load.
 *   DRIFT  (Listing 1): L.   x += x'L; y += y'L; s += L sqrt(1 + x'^2 + y'^2)
 *   MATRIX (G3): R (36 doubles, row-major R[6r+c]), C (6 doubles or NULL = 0).
 *                                   v <- C + R v, each row accumulated from C[r] over c = 0..5 with FMAs
 *   MATRIX2 (track_particles M2; G31): R, C as MATRIX and T (126 doubles, T[21 i + q], q
 *                                   numbering the pairs (j,k), j <= k, as (0,0) (0,1) .. (0,5) (1,1) .. (5,5)).
 *                                   v_i <- C_i + sum_j R_ij v_j + sum_{j<=k} T_ijk v_j v_k; row i accumulated from
 *                                   C_i with FMAs, R terms first (j ascending), then T terms (q ascending) on the
 *                                   rounded products v_j v_k
 *   MATRIX3 (track_particles M3; G35): MATRIX2 plus U (336 doubles, U[56 i + t], t numbering the
 *                                   triples (j,k,l), j <= k <= l, lexicographically): + sum U_ijkl v_j v_k v_l, the
 *                                   terms after the T terms, t ascending, on the products (v_j v_k) v_l.  Always runs
 *                                   in the long-run kernel (12 parameter slots)
 *   RFKICK (G8): V [V], f [Hz], phi [rad].
 *                                   delta += V/(beta0 p0c) sin(phi + 2 pi f (s - s_ref)/(beta0 c)),
 *                                   s_ref = design path length in front of the element on this turn, or with
 *                                   fiducial = 1 (the reduction of PAPER.md:154; G36) s_design + the exactly
 *                                   accumulated mean of s - s_design over the live particles
 *   RCOL   (G17): ax, ay [m].  survive iff |x| <= ax and |y| <= ay
 *   ECOL   (G17): ax, ay [m] semi-axes.  survive iff (x/ax)^2 + (y/ay)^2 <= 1
 *   WAKE   (G9-G16): nb bins, window mode (+ t_lo_rel, dt if EXPLICIT), wake kind with
 *                                   (f, Q, Rs) or (table, n_table, dt_table), interp (1 = linear between
 *                                   bin centres, 0 = own bin)
 *   HISTO: nb, window, t_lo_rel, dt: time histogram only (diagnostic), no kick
 *   TRWAKE (track_through_trwake; G32-G34): fields as WAKE, wake kind RESONATOR_T (f, Q, Rs in
 *                                   Ohm/m) or TABLE [V/C/m].  Per time bin the dipole sums Dx = sum x, Dy = sum y
 *                                   (accumulated exactly in 64-bit fixed point, G33), Vx_i = q sum_{j<=i} Dx_j W_{i-j},
 *                                   x' += Vx(t)/(beta0 p0c), y' += Vy(t)/(beta0 p0c), interpolated as for WAKE.
 *                                   Stage outputs: counts -> hist_out; Dx, Dy, Vx, Vy (4 nb doubles) -> V_out
 */
typedef struct {
    int32_t type;
    int32_t nb;
    int32_t window;
    int32_t wake;
    int32_t interp;
    int32_t fiducial;   /* RFKICK: 1 = phase reference on the bunch's mean path length (G36), 0 = design orbit (G8) */
    double L;
    double V, f, phi;
    double ax, ay;
    double Q, Rs;
    double t_lo_rel, dt, dt_table;
    const double* R;
    const double* C;
    const double* table;
    int64_t n_table;
    const double* T;
    const double* U;
} elg_element;

typedef struct elg_bunch elg_bunch;
typedef struct elg_beamline elg_beamline;

/* Options of elg_track.  All pointers are HOST pointers (nullable); when any is non-NULL the call
 * synchronises the stream before returning.
 *   records : capacity_records x 43 doubles, one record = n_alive, centroid[6], Sigma[36] row-major
 *             (population central moments over live particles, G20); taken after every turn
 *             (ELG_MOM_TURN) or after every element (ELG_MOM_ELEMENT, G26).  n_records returns the number
 *             of records taken (may exceed the capacity; the excess is dropped).
 *   hist_out / V_out / window_out : per-stage outputs of the successive WAKE / HISTO / TRWAKE executions (counts
 *             uint32[nb]; V double[nb] for a WAKE, Dx, Dy, Vx, Vy (4 nb doubles) for a TRWAKE; window = t_lo, dt,
 *             1/dt), used by the stage-by-stage parity protocol; *_written return the totals (in entries / triples).
 */
/* elg_track_opts.flags.  ELG_TRACK_SPARSE_MATRICES: a MATRIX whose entries outside the zero pattern of an uncoupled
 * element (rows x, x': columns x, x', delta; rows y, y': columns y, y', delta; row s: all; row delta: columns s, delta) are
 * exactly zero is applied with the 20 FMAs of that pattern instead of 36.  For finite coordinates the result equals
 * the dense one (up to the sign of a zero); NaN / inf coordinates do not propagate through the skipped terms.  Off by
 * default: the measured configuration applies every matrix densely. */
enum { ELG_TRACK_SPARSE_MATRICES = 1 };

typedef struct {
    int32_t moments_every;
    int32_t flags;               /* ELG_TRACK_* bits, 0 = none */
    double* records;
    int64_t capacity_records;
    int64_t n_records;
    uint32_t* hist_out;
    int64_t hist_capacity;
    int64_t hist_written;
    double* V_out;
    int64_t V_capacity;
    int64_t V_written;
    double* window_out;
    int64_t window_capacity;
    int64_t window_written;
} elg_track_opts;

/* ---- library ---------------------------------------------------------------------------------- */
const char* elg_version(void);
const char* elg_last_error(void);
/* number of kernels this library has launched in this process (for bench.py's gpu_launches) */
int64_t elg_launch_count(void);

/* ---- particle store geometry ------------------------------------------------------------------ */
/* elements between successive arrays of the store: n0 rounded up to a multiple of 32 (256 bytes) */
int64_t elg_soa_stride(int64_t n0);
/* 7 * stride * 8 */
int64_t elg_soa_bytes(int64_t n0);

/* ---- beamline (host only; needs no device) ----------------------------------------------------- */
/* Validates and copies n_elems elements (L finite, apertures > 0, nb >= 2, Q > 1/2, ...).  On a bad
 * element returns ELG_EINVAL and elg_last_error() names its index.  ring = 1: the line closes on itself,
 * RF phase references and EXPLICIT windows advance by the line length every turn (G8).  ring = 0: a line; a bunch
 * sent through it again (n_turns > 1 or a second elg_track) enters it afresh: the references of turn 0 are used on
 * every pass (the turn number still counts up in the lost log).  The design path
 * length is the sequential fp64 sum of L (DRIFT) and C[4] (MATRIX, MATRIX2, MATRIX3) of the preceding elements. */
int32_t elg_beamline_load(elg_beamline** out, const elg_element* h_elems, int64_t n_elems, int32_t ring);
void    elg_beamline_destroy(elg_beamline*);
int64_t elg_beamline_n_elements(const elg_beamline*);
double  elg_beamline_length(const elg_beamline*);
/* design path length in front of element k (0 <= k <= n_elems) on turn 0 */
double  elg_beamline_s_design(const elg_beamline*, int64_t k);
/* number of kernel launches one turn takes under the given moments mode (fused runs, north_star part 1) */
int64_t elg_beamline_launches_per_turn(const elg_beamline*, int32_t moments_every);

/* ---- bunch ------------------------------------------------------------------------------------- */
/* Workspace size for a bunch of n0 particles tracked through bl (nullable: sized for nb <= 65536 and
 * tables <= 65536 points), with room for lost_capacity lost-particle records (0 = none kept). */
int32_t elg_workspace_bytes(int64_t n0, const elg_beamline* bl, int64_t lost_capacity, int64_t* bytes);
/* Borrow d_soa (layout above; already filled by the caller, or to be filled by elg_bunch_upload) and
 * d_work (256-byte aligned, work_bytes >= elg_workspace_bytes(n0, sized_for, lost_capacity); sized_for is
 * only read during this call).  p0c_eV, mc2_eV: reference momentum and
 * rest energy (G7); charge_C: bunch charge, macro-charge q = charge / n0 for the whole run (G15).
 * stream: a cudaStream_t (NULL = default stream).  n_alive = n0, turn = 0, lost log empty. */
int32_t elg_bunch_create(elg_bunch** out, int64_t n0, void* d_soa, void* d_work, int64_t work_bytes,
                         const elg_beamline* sized_for, int64_t lost_capacity, double p0c_eV, double mc2_eV, double charge_C, void* stream);
void    elg_bunch_destroy(elg_bunch*);
/* Copy n0 particles from host arrays (pinned or pageable) into the store and rewind the bunch.
 * h_ids NULL: ID = index (G27). */
int32_t elg_bunch_upload(elg_bunch*, const double* const h_coords[6], const int64_t* h_ids);
/* The caller has rewritten d_soa with n0 fresh particles: n_alive = n0, turn = 0, lost log empty. */
int32_t elg_bunch_rewind(elg_bunch*);

/* Track n_turns passes through the beamline.  opts nullable.  Asynchronous on the bunch's stream unless
 * opts asks for host outputs.  Every kernel is launched with the programmatic-stream-serialization attribute and begins
 * with griddepcontrol.wait, so the order is the stream's.  Environment switches for A/B measurements (read once per
 * process; the defaults are the measured best): ELG_PDL=0 (plain launches), ELG_CHAIN_RING=0 (short DRIFT / MATRIX runs
 * through chain_kernel instead of the bulk-copy ring), ELG_HIST_AGGREGATE=1, ELG_CHAIN_P=2|4. */
int32_t elg_track(elg_bunch*, const elg_beamline*, int64_t n_turns, elg_track_opts* opts);

/* CUDA graphs.  elg_track (and elg_bunch_rewind) may be CAPTURED by the caller (cudaStreamBeginCapture on the bunch's
 * stream; the stream must not be the legacy default stream) when opts asks for no host output, profiling is off and
 * the beamline has been tracked once before (wake tables are uploaded on first use): nothing in the call synchronises
 * or reads the device; inside a capture elg_track clears the compaction's tile status and restarts its epoch first.
 * A replay repeats the captured launches with the parameters of the capture (buffers, turn numbers, RF phase
 * references, record slots), so it is valid whenever the bunch is in the state the capture started from -- normally the
 * capture begins with the caller's copy of fresh particles into d_soa and elg_bunch_rewind.  The library's HOST mirror of
 * the device state (current store, count slot, epoch, turn, records in the device ring) is advanced by the capture, not
 * by a replay: save it after the capture and restore it after every replay before calling anything else on the bunch.
 * Records of a captured run stay in the device ring (the host copy needs opts->records, which cannot be captured). */
int32_t elg_bunch_host_state_save(const elg_bunch*, int64_t state[8]);
int32_t elg_bunch_host_state_restore(elg_bunch*, const int64_t state[8]);

/* elg_bunch_upload followed by elg_track in ONE call with the upload pipelined against the tracking: the bunch is
 * cut into n_chunks particle ranges (n_chunks <= 1: no pipelining; at most 32 are used); each range is copied from the HOST arrays on a
 * copy stream owned by the bunch and, as soon as it has landed, the leading per-particle maps of the first turn
 * (everything in front of the first WAKE / HISTO / TRWAKE, aperture, bunch-fiducial RFKICK or per-element record)
 * run on that range while the following ranges are still being copied.  Results are identical to
 * elg_bunch_upload + elg_track.  Host arrays as for elg_bunch_upload (pinned memory for real overlap); they must
 * stay valid until the bunch's stream has been synchronised. */
int32_t elg_upload_and_track(elg_bunch*, const elg_beamline*, const double* const h_coords[6], const int64_t* h_ids,
                             int64_t n_turns, elg_track_opts* opts, int32_t n_chunks);

/* Moments of the live particles now (north_star part 4).  n_alive == 0: ELG_ESTATE, outputs untouched. */
int32_t elg_moments(elg_bunch*, int64_t* n_alive, double h_centroid[6], double h_sigma[36]);
/* Lost-particle log in canonical order (G18): chronological (turn, element index), then original array
 * position.  coords6 is cap x 6 row-major (the coordinates at the aperture; its s is the loss position),
 * nullable.  cap < n_lost: fills cap records and returns ELG_ECAPACITY with the true n_lost. */
int32_t elg_lost(elg_bunch*, int64_t* n_lost, int64_t cap, int64_t* h_ids, int32_t* h_turn, int32_t* h_elem,
                 double* h_coords6);
int32_t elg_n_alive(elg_bunch*, int64_t* n_alive);
/* Copy the live particles to host arrays of capacity cap each (any pointer nullable). */
int32_t elg_bunch_read(elg_bunch*, double* const h_coords[6], int64_t* h_ids, int64_t cap);
/* Device pointer of coordinate c (0..5) or of the IDs (c = 6) in the CURRENT store (compaction ping-pongs
 * between d_soa and a copy in the workspace). */
int32_t elg_bunch_device_array(elg_bunch*, int32_t c, void** d_ptr);

/* ---- per-kernel device timing (for bench.py's roofline object) ---------------------------------------
 * With profiling on, every kernel the bunch launches is bracketed by a pair of CUDA events on the bunch's
 * stream.  elg_profile_read synchronises the stream, returns per kernel kind the number of launches and
 * their summed device time since the last read (h_launches, h_ms: ELG_K_COUNT entries each) and resets
 * the counters.  h_bytes / h_flops (nullable): the ALGORITHMIC work of those launches per kind -- bytes = 8 x (coordinates
 * the run reads + coordinates it writes) x live particles of the launch (+ 16 for the IDs of a compacting run, which
 * moves all seven arrays), flops = the per-particle flop counts of DESIGN.md section 5 x live particles -- accumulated
 * on the device from the live count each launch sees (the host never knows it).  Off by default. */
enum { ELG_K_CHAIN = 0, ELG_K_CHAIN_COMPACT = 1, ELG_K_WINDOW = 2, ELG_K_HIST = 3, ELG_K_WAKE_SAMPLES = 4,
       ELG_K_CONV = 5, ELG_K_MOMENTS = 6, ELG_K_CHAIN_LONG = 7, ELG_K_COUNT = 8 };
int32_t elg_profile_enable(elg_bunch*, int32_t on);
int32_t elg_profile_read(elg_bunch*, int64_t* h_launches, double* h_ms, double* h_bytes, double* h_flops);

/* ---- single-stage test hooks (not the user boundary) -------------------------------------------------
 * For the stage-by-stage parity protocol (the paper compares CPU and GPU element by element on the
 * same inputs).  The bunch-based hooks run ONE stage of elg_track on the particles currently in
 * the bunch -- upload the oracle's input of that stage with elg_bunch_upload first -- through the same planner code
 * and therefore the same kernels, instantiations and launch configurations as tracking itself:
 *   elg_dbg_histogram         min/max epilogue run, window_kernel (EXPLICIT window t_lo, dt), hist_kernel with the
 *                             occupied-range privatisation -> counts (uint32[nb], DEVICE)
 *   elg_dbg_dipole_histogram  the same with dipole_hist_kernel + dipole_finalize_kernel -> counts, Dx[nb] Dy[nb] (G33)
 *   elg_dbg_kick / _tkick     window as above, then the wake kick as tracking applies it: OP_KICK / OP_TKICK as a
 *                             fused run of one op reading V (or Vx, Vy) copied from the caller's DEVICE arrays (G14)
 *   elg_dbg_compact           a run of zero maps ending in the aperture: predicate + stable compaction + lost log
 *                             (PAPER.md:141 loss contract); read the result with elg_bunch_read / elg_lost
 * nb must not exceed the bin capacity the workspace was sized for.  The two array-based hooks run the wake-sample and
 * convolution kernels of tracking on caller-supplied DEVICE arrays (whole bin range). */
int32_t elg_dbg_histogram(elg_bunch*, double t_lo, double dt, int32_t nb, uint32_t* d_counts);
int32_t elg_dbg_dipole_histogram(elg_bunch*, double t_lo, double dt, int32_t nb, uint32_t* d_counts, double* d_D);
int32_t elg_dbg_kick(elg_bunch*, double t_lo, double dt, int32_t nb, const double* d_V, int32_t interp);
int32_t elg_dbg_tkick(elg_bunch*, double t_lo, double dt, int32_t nb, const double* d_Vx, const double* d_Vy,
                      int32_t interp);
int32_t elg_dbg_compact(elg_bunch*, int32_t type /* ELG_RCOL | ELG_ECOL */, double ax, double ay);
/* the fp64 roofline denominator, measured: a DFMA-only kernel (8 independent chains per thread, register operands, two
 * blocks of 256 threads per SM) timed with CUDA events; d_scratch: >= 2048 bytes of DEVICE memory; iters: loop trips of
 * 128 DFMA per thread.  Returns 2 x DFMA/s in TFLOP/s and the kernel time. */
int32_t elg_dbg_fp64_peak(double* d_scratch, int64_t iters, double* h_tflops, double* h_ms, void* stream);
int32_t elg_dbg_wake_samples(int32_t kind, int32_t nb, double dt, double f, double Q, double Rs,
                             const double* d_table, int64_t n_table, double dt_table, double* d_W, void* stream);
int32_t elg_dbg_convolve(const uint32_t* d_counts, const double* d_W, int32_t nb, double q, double* d_V,
                         void* stream);

/* ---- an entry point that allocates nothing ------------------------------------------------------------------------
 * The dipole histogram stage (TRWAKE, G32-G33: bin counts and the exact per-bin sums of x and y) for callers that cannot
 * call cudaMalloc and have no workspace to lend: code under CUDA-graph capture, tight serving loops, harnesses that
 * forbid allocation.  Inputs and outputs are the caller's DEVICE arrays: s, x, y (n doubles each, 16-byte aligned),
 * counts (uint32[nb]), D (double[2 nb]: Dx then Dy); bin k = [t_lo + k dt, t_lo + (k + 1) dt) of t = s inv_bc (G9, G10).
 * The scratch of the stage (a state block + four 64-bit accumulators per bin) is a file-scope device array inside the
 * library, 524 800 bytes, held by every GPU that loads the library until the process exits; hence
 * nb <= elg_noalloc_max_bins() = 16384, beyond which the call returns ELG_ECAPACITY and launches nothing.
 * The call performs no cudaMalloc / cudaFree and calls no allocating library routine; it launches three kernels on
 * `stream` (the histogram and finalize kernels are tracking's own) and does not synchronise.  Results equal
 * elg_dbg_dipole_histogram's bit for bit.
 * Every call on a device shares the one array, which keeps the last call's contents: each call clears what must start
 * at zero (accumulators, counts) itself, and calls that OVERLAP on the GPU (two streams without an ordering between
 * them, two host threads) race on it -- serialise them. */
int32_t elg_noalloc_max_bins(void);
int32_t elg_dipole_histogram_noalloc(const double* d_s, const double* d_x, const double* d_y, int64_t n, double inv_bc,
                                     double t_lo, double dt, int32_t nb, uint32_t* d_counts, double* d_D, void* stream);

#ifdef __cplusplus
}
#endif
#endif
