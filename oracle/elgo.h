/* elgo.h -- CPU ORACLE for the macroparticle tracking hot path of arXiv:1710.07350.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference leg may build, load or call anything under oracle/.
 * It shares no code with the CUDA path (paper_1710_07350_b200/): no headers, helpers, tables or
 * constants.  It is a plain, slow, sequential fp64 restatement of what the path computes, written so
 * that it can be checked against the paper by eye.  Citations "PAPER.md:NN" are lines of
 * /root/reference/PAPER.md; "Gk" are the readings listed in DESIGN.md ("Readings of the paper").
 *
 * Parity status of each function (what pins it, see tests/test_oracle_pins.py):
 *   elgo_drift        pinned  - Listing 1 exact cases, literal re-evaluation
 *   elgo_matrix       pinned  - closed forms, identity, inverse, symplectic invariants
 *   elgo_matrix3      pinned  - U = 0 equals elgo_matrix2 bitwise, one-entry index pins, thin octupole closed form,
 *                               third-order path length of a drift
 *   elgo_matrix2      pinned  - T = 0 equals elgo_matrix bitwise, one-entry index pins, thin sextupole and
 *                               second-order drift closed forms (exact drift to O(x'^4))
 *   elgo_rfkick       pinned  - crest/zero-crossing/periodicity/slope closed forms
 *   elgo_fiducial     pinned  - plain mean against math.fsum, kicks invariant under a common delay
 *   elgo_aperture     pinned  - hand-placed particles, brute-force stable partition, erf fractions
 *   elgo_window/histogram  pinned - hand-placed bins, edge rule, sum of counts
 *   elgo_wake_samples pinned  - beam-loading theorem, independent evaluation
 *   elgo_convolve     pinned  - brute-force double loop, numpy.convolve, continuous closed form
 *   elgo_convolve_resonator  pinned - equals elgo_convolve of elgo_wake_samples (<= 1e-12 of the maximum)
 *   elgo_kick         pinned  - bin-centre / midpoint / clamped cases
 *   elgo_dipole_histogram, elgo_convolve_d, elgo_tkick (TRWAKE)  pinned - plain weighted sums (math.fsum), brute-force
 *                               convolution, two-particle closed form, zero offset => zero kick, linearity, kick at a
 *                               bin centre / midpoint / beyond the end centres / own bin
 *   elgo_lost         pinned  - hand-placed losses, canonical order, cap < n_lost truncation
 *   elgo_track record placement (ELGO_MOM_ELEMENT / ELGO_MOM_TURN, G26)  pinned - three-particle hand case, 77 records
 *                               for cfg1; ring flag (G8): RF reference advances per turn on a ring only
 *   elgo_moments      pinned  - symmetric hand sets, shift invariance, Gaussian statistics
 *   elgo_track        pinned  - equals the composition, by hand, of the pinned stage functions in the order of
 *                               PAPER.md:51 (test_track_is_the_composition_of_stages, test_trwake_track_is_...),
 *                               turn advance and thread-count invariance, loss sequence of a small cfg4, record
 *                               placement (above).  The paper prints no end-to-end values for whole beamlines, so
 *                               nothing beyond the composition can be pinned to it.
 *
 * Precision: the paper computes in double precision; so does the oracle.  Sums
 * (convolution, moments) are accumulated in long double so that the oracle is closer to the exact
 * value than any fp64 summation order.  The per-particle maps use std::fma in a fixed order (the
 * "arithmetic specification") and the file is compiled with -ffp-contract=off.
 */
#ifndef ELGO_H
#define ELGO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { ELGO_OK = 0, ELGO_EINVAL = -1, ELGO_ENOMEM = -2, ELGO_ESTATE = -4, ELGO_ECAPACITY = -5 };

/* element types (names: PAPER.md:175 glossary; north_star) */
enum { ELGO_DRIFT = 1, ELGO_MATRIX = 2, ELGO_RFKICK = 3, ELGO_RCOL = 4, ELGO_ECOL = 5,
       ELGO_WAKE = 6, ELGO_HISTO = 7, ELGO_MATRIX2 = 8, ELGO_TRWAKE = 9, ELGO_MATRIX3 = 10 };
/* histogram window modes (G10) */
enum { ELGO_WIN_EXPLICIT = 0, ELGO_WIN_AUTO_MINMAX = 1, ELGO_WIN_AUTO_TABLE = 2 };
/* wake kinds (G12) */
enum { ELGO_WAKE_RESONATOR = 0, ELGO_WAKE_TABLE = 1, ELGO_WAKE_RESONATOR_T = 2 /* transverse, G34 */,
       ELGO_WAKE_RESONATOR_REC = 3 /* longitudinal resonator by the O(nb) two-term recurrence, G37 */ };
/* when elgo_track records moments (G26) */
enum { ELGO_MOM_NONE = 0, ELGO_MOM_TURN = 1, ELGO_MOM_ELEMENT = 2 };

/* One beamline element.  Unused fields are ignored.
 *   DRIFT : L
 *   MATRIX: R (36, row-major R[6*r+c]), C (6, may be NULL = 0)
 *   MATRIX2: R, C as MATRIX, T (126 = 6 x 21, T[21*i + q], q numbers the pairs (j,k), j <= k, in the order
 *           (0,0) (0,1) .. (0,5) (1,1) .. (5,5)): second-order transport map (G31)
 *   MATRIX3: MATRIX2 plus U (336 = 6 x 56, U[56*i + t], t numbers the triples (j,k,l), j <= k <= l, in
 *           lexicographic order): third-order transport map (G35)
 *   RFKICK: V [V], f [Hz], phi [rad], fiducial
 *   RCOL  : ax, ay [m]      ECOL: ax=a, ay=b [m]
 *   WAKE  : nb, window, (t_lo_rel, dt if EXPLICIT), wake kind, (f, Q, Rs) or (table, n_table, dt_table), interp
 *   HISTO : nb, window, t_lo_rel, dt   (histogram only, no kick)
 *   TRWAKE: as WAKE, wake kind RESONATOR_T or TABLE [V/C/m]: transverse (dipole) wake, kicks x' and y' (G32-G34)
 */
typedef struct {
    int32_t type;
    int32_t nb;
    int32_t window;
    int32_t wake;
    int32_t interp;
    int32_t fiducial;   /* RFKICK: 1 = phase reference on the bunch's mean path length (G36), 0 = design (G8) */
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
} elgo_element;

typedef struct elgo_bunch elgo_bunch;
typedef struct elgo_beamline elgo_beamline;

/* ---- stage functions on plain arrays (used stage by stage in the parity protocol) ---- */
void   elgo_drift(double* x, const double* xp, double* y, const double* yp, double* s, int64_t n, double L);
void   elgo_matrix(double* const v[6], int64_t n, const double* R36, const double* C6);
/* second-order map: v_i <- C_i + sum_j R_ij v_j + sum_{j<=k} T_ijk v_j v_k (G31) */
void   elgo_matrix2(double* const v[6], int64_t n, const double* R36, const double* C6, const double* T126);
/* third-order map (G35): ... + sum_{j<=k<=l} U_ijkl v_j v_k v_l */
void   elgo_matrix3(double* const v[6], int64_t n, const double* R36, const double* C6, const double* T126,
                    const double* U336);
/* G36: s_design + (plain long-double sum of the rounded differences s_i - s_design) / n; n = 0: s_design */
double elgo_fiducial(const double* s, int64_t n, double s_design);
void   elgo_rfkick(const double* s, double* delta, int64_t n, double A, double omega, double phi0,
                   double s_ref, double inv_bc);
/* survive[i] = 1/0.  kind = ELGO_RCOL or ELGO_ECOL. */
void   elgo_aperture_flags(const double* x, const double* y, int64_t n, int32_t kind, double ax, double ay,
                           uint8_t* survive);
/* stable partition of the first n entries of 6 coordinate arrays + ids by survive[]; returns n_surv.
   lost_* receive the lost particles in increasing position order (capacity n each; lost_v is 6 arrays). */
int64_t elgo_compact(double* const v[6], int64_t* id, int64_t n, const uint8_t* survive,
                     double* const lost_v[6], int64_t* lost_id);
/* window: out[0]=t_lo, out[1]=dt, out[2]=inv_dt.  t_design is used by EXPLICIT only. */
int32_t elgo_window(const double* s, int64_t n, double inv_bc, int32_t mode, int32_t nb,
                    double t_lo_rel, double dt_in, double t_design, double out[3]);
/* counts[nb] (zeroed here); bin_of[i] (nullable) receives the bin or -1. returns number binned */
int64_t elgo_histogram(const double* s, int64_t n, double inv_bc, double t_lo, double inv_dt, int32_t nb,
                       uint32_t* counts, int32_t* bin_of);
int32_t elgo_wake_samples(int32_t kind, int32_t nb, double dt, double f, double Q, double Rs,
                          const double* table, int64_t n_table, double dt_table, double* W);
void   elgo_convolve(const uint32_t* counts, const double* W, int32_t nb, double q, double* Vout);
/* the same V for the resonator wake of G12 by the O(nb) complex recurrence (G37), no W array */
int32_t elgo_convolve_resonator(const uint32_t* counts, int32_t nb, double q, double dt, double f, double Q, double Rs,
                                double* Vout);
/* TRWAKE (G32-G34): counts[nb] and the per-bin dipole sums Dx[nb], Dy[nb] = sum of x, y of the particles in the
   bin, accumulated sequentially in long double (G33: the plain definition; particles out of range are counted only) */
int64_t elgo_dipole_histogram(const double* s, const double* x, const double* y, int64_t n, double inv_bc, double t_lo,
                              double inv_dt, int32_t nb, uint32_t* counts, double* Dx, double* Dy);
/* V_i = q sum_{j<=i} D_j W_{i-j} (G13 with real weights) */
void   elgo_convolve_d(const double* D, const double* W, int32_t nb, double q, double* Vout);
/* x' += Vx(t)/(beta0 p0c), y' += Vy(t)/(beta0 p0c), interpolation as elgo_kick (G14) */
void   elgo_tkick(const double* s, double* xp, double* yp, int64_t n, double inv_bc, double t_lo, double inv_dt,
                  int32_t nb, const double* Vx, const double* Vy, double inv_E, int32_t interp);
void   elgo_kick(const double* s, double* delta, int64_t n, double inv_bc, double t_lo, double inv_dt,
                 int32_t nb, const double* V, double inv_E, int32_t interp);
/* n>0 required. centroid[6], sigma[36] row-major, population (1/n) central moments (G20). */
int32_t elgo_moments(const double* const v[6], int64_t n, double centroid[6], double sigma[36]);

/* ---- derived constants (arithmetic specification) ---- */
double elgo_beta0(double p0c_eV, double mc2_eV);          /* p0c / sqrt(p0c^2 + mc2^2)  */
double elgo_inv_bc(double beta0);                          /* 1 / (beta0 * c)            */
double elgo_inv_E(double beta0, double p0c_eV);            /* 1 / (beta0 * p0c)          */

/* ---- bunch / beamline / tracking (same call shapes as the C-ABI of include/elg.h, host memory) ---- */
int32_t elgo_bunch_create(elgo_bunch** out, int64_t n0, const double* const coords[6], const int64_t* ids,
                          double p0c_eV, double mc2_eV, double charge_C);
void    elgo_bunch_destroy(elgo_bunch*);
/* ring = 1: RF phase references and EXPLICIT windows advance by the line length every turn (G8); ring = 0: every pass
 * uses the references of turn 0 (a line is entered afresh) */
int32_t elgo_beamline_load(elgo_beamline** out, const elgo_element* elems, int64_t n_elems, int32_t ring);
void    elgo_beamline_destroy(elgo_beamline*);
/* design path length (G8) in front of element k on turn 0, and the ring/line length */
double  elgo_beamline_s_design(const elgo_beamline*, int64_t k);
double  elgo_beamline_length(const elgo_beamline*);

typedef struct {
    int32_t moments_every;       /* ELGO_MOM_*                                             */
    int32_t n_threads;           /* >1: per-particle loops split over threads (same results) */
    double* records;             /* nullable; capacity_records x 43 doubles: n, C[6], Sigma[36] */
    int64_t capacity_records;
    int64_t n_records;           /* out */
    uint32_t* hist_out;          /* nullable; histograms of successive WAKE/HISTO executions, nb each */
    int64_t hist_capacity;       /* in uint32 entries */
    int64_t hist_written;        /* out */
    double* V_out;               /* nullable; V arrays of successive WAKE executions; a TRWAKE appends Dx, Dy, Vx, Vy */
    int64_t V_capacity;
    int64_t V_written;           /* out */
    double* window_out;          /* nullable; (t_lo, dt, inv_dt) of successive WAKE/HISTO executions */
    int64_t window_capacity;     /* in triples */
    int64_t window_written;      /* out */
} elgo_track_opts;

int32_t elgo_track(elgo_bunch*, const elgo_beamline*, int64_t n_turns, elgo_track_opts* opts);
int64_t elgo_n_alive(const elgo_bunch*);
int32_t elgo_bunch_read(const elgo_bunch*, double* const coords[6], int64_t* ids, int64_t cap);
int32_t elgo_moments_now(const elgo_bunch*, int64_t* n_alive, double centroid[6], double sigma[36]);
/* lost log in canonical order (G18): chronological (turn, element), then original position */
int32_t elgo_lost(const elgo_bunch*, int64_t* n_lost, int64_t cap, int64_t* ids, int32_t* turn, int32_t* elem,
                  double* coords6 /* cap x 6 row-major, nullable */);

#ifdef __cplusplus
}
#endif
#endif
