// elg_kernels.cuh -- device code of libelg (sm_100a).  Hand-written CUDA; no code shared with oracle/.
//
// Arithmetic specification: every per-particle map is written with explicit
// fma() in a fixed order and the file is compiled with -fmad=false, so nothing else is contracted.
// IEEE fma / sqrt / div are correctly rounded on the device, hence DRIFT, MATRIX, aperture predicates,
// window and bin indices are bit-reproducible; only sin/cos/exp (<= 2 ulp) and summation order differ
// from a sequential CPU evaluation.
//
// Kernels (one section each):
//   chain_kernel, chain_long_kernel    fused run of element maps (short HBM-bound runs / long fp64-bound runs)
//   compact_kernel                 fused run ending in an aperture + stable single-pass stream compaction
//   window_kernel                  min/max partials -> histogram window + occupied bin range, zero counts
//   hist_kernel                    shared-memory privatised time histogram
//   wake_samples_kernel, conv_kernel   wake function samples and causal convolution
//   moments_kernel                 shifted one-pass deterministic fp64 tree reduction (27 sums)
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace elg {

constexpr int kBlock = 256;            // threads per block
constexpr int kWarps = kBlock / 32;
constexpr int kP = 2;                  // particles per thread = one 128-bit access per coordinate
constexpr int kTile = kBlock * kP;     // particles per tile
constexpr int kHistSmemBins = 16384;   // 64 KB of privatised bins per block
constexpr int kNMom = 27;              // 6 first + 21 second shifted sums
// long-run kernel geometry of the higher-order levels (threads per block, particles per thread, register cap)
#ifndef ELG_L0_NT
#define ELG_L0_NT 384
#define ELG_L0_PL 6
#define ELG_L0_REGS 168          // the most 384 threads can have: 152 suffice, but with 168 ptxas schedules the DFMA chains 4 % faster
#endif
#ifndef ELG_L3_REGS
#define ELG_L3_REGS 168
#endif
#ifndef ELG_L1_NT
#define ELG_L1_NT 256
#define ELG_L1_PL 6
#define ELG_L1_REGS 200
#endif
#ifndef ELG_MM_ROWS
#define ELG_MM_ROWS 2            // rows of a MATRIX formed together in the long-run kernel (levels 0, 2, 3)
#endif
#ifndef ELG_MM_ROWS_L3
#define ELG_MM_ROWS_L3 0         // ... at level 3 (dense matrices between the zero-pattern ones of the flagged option); 0: chain after chain
#endif
#ifndef ELG_MM_ROWS_L1
#define ELG_MM_ROWS_L1 1         // ... at level 1 (second-order maps)
#endif
#ifndef ELG_TKICK_BASE
#define ELG_TKICK_BASE 1         // 1: the base (fully unrolled) chain_kernel instantiations also hold the transverse wake kick
#endif
#ifndef ELG_BIN_MAGIC
#define ELG_BIN_MAGIC 1          // bin_of: floor by adding 1.5 x 2^52 instead of FRND / F2I (0: conversions)
#endif
#ifndef ELG_L2_NT
#define ELG_L2_NT 384
#define ELG_L2_PL 4
#define ELG_L2_REGS 144
#endif

enum : uint8_t { OP_DRIFT = 1, OP_MATRIX = 2, OP_RFKICK = 3, OP_KICK = 4,
                 OP_MATRIX2 = 5,      // second-order map: this slot holds R, C; the next three hold T (OP_CONT)
                 OP_CONT = 6,
                 OP_TKICK = 7,        // transverse wake kick of the preceding TRWAKE (G32)
                 OP_MATRIX3 = 8,      // third-order map: R, C | 3 slots Tt[21][6] | 8 slots Ut[56][6] (12 slots, G35)
                 OP_MATRIX_UNC = 9,   // MATRIX whose zero pattern is that of an uncoupled element (flagged option)
                 OP_KICK3 = 10 };     // OP_KICK + OP_TKICK of an RFCW composite (same binning): one bin look-up for both
enum { AP_NONE = 0, AP_RCOL = 1, AP_ECOL = 2 };

// Device-resident tracking state (first bytes of the workspace).  Nothing here is read by the host
// during elg_track: n_alive never crosses PCIe on the hot path (the paper syncs per lossy element,
// PAPER.md:141 step 2).
struct DevState {
    long long n_alive[2];      // ping-pong: a compaction reads slot cur, writes slot cur^1
    long long n_lost[2];
    double win[4];             // t_lo, dt, inv_dt, -
    double smin, smax;         // exact min / max of s over live particles
    long long bin_lo, bin_hi;  // occupied bin range (clamped to [0, nb-1]); bin_lo > bin_hi: nothing binned
    unsigned int tile_counter; // dynamic tile ids for the look-back scan
    unsigned int done_counter;
    unsigned int mom_done;
    unsigned int fid_done;
    unsigned long long fid_acc[2];   // exact fixed-point sum of s - s_design (G36)
    double s_ref;              // fiducial path length of the bunch, read by RFKICK ops with the fiducial flag
    long long zero_bits;       // always 0: a value the compiler cannot see through (matrix_map_uniform)
    unsigned long long work[16];     // per kernel kind (ELG_K_*): algorithmic bytes, flops of the launches since the last
                                     // elg_profile_read (only counted while profiling is on)
};

// work accounting for elg_profile_read: one thread adds what this launch moves and computes, from the live count
// the launch itself sees (the host never knows it).  kind < 0: profiling off.
__device__ __forceinline__ void account_work(DevState* st, int kind, long long n, unsigned int bytes_pp, unsigned int flops_pp) {
    if (kind >= 0 && blockIdx.x == 0 && threadIdx.x == 0 && n > 0) {
        atomicAdd(&st->work[2 * kind], (unsigned long long)n * bytes_pp);
        atomicAdd(&st->work[2 * kind + 1], (unsigned long long)n * flops_pp);
    }
}

struct ChainCommon {
    double* src[6];
    double* dst[6];
    long long* id_src;
    long long* id_dst;
    DevState* st;
    int cur;                   // n_alive / n_lost slot to read
    int n_ops;
    unsigned int rmask, wmask; // coordinates loaded / stored (accessor rule)
    int ap_type;               // AP_*
    double ap_x, ap_y;         // RCOL: ax, ay.  ECOL: 1/a, 1/b
    long long* lost_id;        // lost log (SoA, capacity lost_cap)
    long long* lost_te;        // turn << 32 | element
    double* lost_v;            // 6 arrays at stride lost_cap
    long long lost_cap;
    long long te_code;
    unsigned long long* tile_status;
    unsigned int epoch;
    int want_minmax;
    double* mm_partial;        // [2 * gridDim.x]
    const double* V;           // OP_KICK operands
    int nb;
    int interp;
    const double* Vx;          // OP_TKICK operands
    const double* Vy;
    int t_nb;
    int t_interp;
    long long range_lo;        // chain kernels work on particles [range_lo, min(range_hi, n_alive)); range_hi < 0: n_alive
    long long range_hi;        // (pipelined upload: one range per chunk, elg_upload_and_track)
    double* mom_partial;       // moment epilogue (MOM instantiations): per-block partials [kNMom][gridDim.x]
    double* mom_record;        //   and the 43-double record to fill (n, centroid, Sigma), a13 / G26
    int prof_kind;             // work accounting (account_work): ELG_K_* or -1
    unsigned int bytes_pp, flops_pp;     // algorithmic bytes / flops of this run per live particle
};

template <int MAXOPS>
struct ChainArgs {
    ChainCommon c;
    uint8_t type[MAXOPS];
    uint8_t mat_run[MAXOPS];               // number of consecutive OP_MATRIX slots starting at this one (host-computed)
    alignas(16) double coef[MAXOPS][42];   // MATRIX: R[36], C[6].  DRIFT: L.  RFKICK: A, omega, phi0, s_ref, inv_bc.
                               // KICK: inv_bc, inv_E.  MATRIX2: R[36], C[6], then 3 slots = Tt[21][6] (pair-major)
};

// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ unsigned long long ld_relaxed(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_relaxed(unsigned long long* p, unsigned long long v) {
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
// streaming 128-bit accesses: every particle is touched once per launch, keep L1 for the tables
__device__ __forceinline__ double2 ld_stream2(const double* p) {
    double2 r;
    asm volatile("ld.global.L1::no_allocate.v2.f64 {%0, %1}, [%2];" : "=d"(r.x), "=d"(r.y) : "l"(p));
    return r;
}
__device__ __forceinline__ double ld_stream1(const double* p) {
    double r;
    asm volatile("ld.global.L1::no_allocate.f64 %0, [%1];" : "=d"(r) : "l"(p));
    return r;
}

// asynchronous copies, mbarriers, named barriers (PTX)
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, int src_bytes) {
    const unsigned int d = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async8(void* smem_dst, const void* gsrc, int src_bytes) {
    const unsigned int d = (unsigned int)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;" ::"r"(d), "l"(gsrc), "r"(src_bytes) : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() { asm volatile("cp.async.wait_all;" ::: "memory"); }
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// mbarrier + 1-D bulk copy (TMA unit, SASS UBLKCP): global -> shared without registers or L1, completion counted in bytes
__device__ __forceinline__ unsigned int smem_u32(const void* p) { return (unsigned int)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned int count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned int bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned long long* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned int parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "MBAR_WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra MBAR_DONE_%=;\n"
        "bra MBAR_WAIT_%=;\n"
        "MBAR_DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gsrc, unsigned int bytes, unsigned long long* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(smem_dst)),
                 "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
template <int ID, int N>
__device__ __forceinline__ void named_barrier() { asm volatile("bar.sync %0, %1;" ::"n"(ID), "n"(N) : "memory"); }

// Programmatic dependent launch: first statement of every kernel.  Kernels are launched with the programmatic-stream-
// serialization attribute (elg.cu, launch_k), which lets a kernel be scheduled while its predecessor in the stream is
// still draining; griddepcontrol.wait then blocks until the predecessor has completed and its writes are visible.  No
// kernel touches global memory before the wait, so the semantics are those of plain stream order; what is gained is
// the launch latency between dependent kernels (the small configurations are launch-bound: cfg0 is 6 launches of 5-20
// us; measured without / with: cfg0 53 -> 43 us, cfg1 1.39 -> 1.29 ms, cfg2 1.72 -> 1.62 ms, cfg4 1.74 -> 1.67 ms).
// No kernel calls griddepcontrol.launch_dependents: with an explicit early trigger the blocks of the next kernels
// become resident while the current one is still working and cfg2 ran 9 % SLOWER than without the attribute.
// A no-op when the kernel was launched without the attribute (ELG_PDL=0).
__device__ __forceinline__ void pdl_begin() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

// bin of a time coordinate (G10): floor((s*inv_bc - t_lo)*inv_dt) in [0, nb) else -1.  For 0 <= u < nb <= 2^24 the
// floor is taken without FRND.F64 / F2I.F64 (quarter-rate conversions): u + 1.5 x 2^52 lies in [2^52, 2^53), where
// doubles are the integers, so the addition rounds u to the nearest integer r, the low word of the sum's bit pattern IS
// r, and floor(u) = r - (r > u).  floor(u) >= 0 <=> u >= 0 and floor(u) < nb <=> u < nb, so the range test is the
// definition's; NaN fails it.
__device__ __forceinline__ int bin_of(double s, double inv_bc, double t_lo, double inv_dt, int nb, double* u_out) {
    const double t = s * inv_bc;
    const double u = (t - t_lo) * inv_dt;
    *u_out = u;
    const bool in_range = (u >= 0.0) && (u < (double)nb);        // NaN: false
#if !ELG_BIN_MAGIC
    return in_range ? (int)floor(u) : -1;
#endif
    constexpr double kMagic = 6755399441055744.0;                // 1.5 x 2^52
    const double m = u + kMagic;                                 // (evaluated for every u, used only in range: no branch)
    const double r = m - kMagic;
    const int k = __double2loint(m) - ((r > u) ? 1 : 0);
    return in_range ? k : -1;
}

// ---------------------------------------------------------------------------------------------------
// Element maps on P particles held in registers.  Coefficients come straight from the kernel parameter
// constant bank (uniform operands of DFMA), so a MATRIX costs 42 DFMA per particle and no LSU traffic.
// One coefficient fetch (LDCU) feeds P DFMAs: P = 4 keeps the fp64 pipe, not the constant path, the
// limiter of long runs (profiles/r01a_first_path.md, round 1).
// ---------------------------------------------------------------------------------------------------
// v -> w through one MATRIX (G3): row r accumulates from C[r] over c = 0..5 with FMAs, in that order.
template <int P>
__device__ __forceinline__ void matrix_map(const double* __restrict__ c, const double (&v)[P][6], double (&w)[P][6]) {
#pragma unroll
    for (int r = 0; r < 6; r++) {
#pragma unroll
        for (int p = 0; p < P; p++) {
            double acc = c[36 + r];
#pragma unroll
            for (int cc = 0; cc < 6; cc++) acc = fma(c[6 * r + cc], v[p][cc], acc);
            w[p][r] = acc;
        }
    }
}

// second-order terms of MATRIX2 (G31): w[p][r] += sum over the pairs q = (j,k), j <= k, of T[r][q] (v_j v_k),
// q ascending, continuing row r's FMA chain after the six first-order terms.  tt = Tt[21][6] (pair-major), so one
// pair costs P products and 6 P DFMA on six coefficients (uniform operands when tt points into the parameter bank).
template <int P>
__device__ __forceinline__ void matrix2_terms(const double* __restrict__ tt, const double (&v)[P][6], double (&w)[P][6]) {
    int q = 0;
#pragma unroll
    for (int j = 0; j < 6; j++) {
#pragma unroll
        for (int k = j; k < 6; k++) {
#pragma unroll
            for (int p = 0; p < P; p++) {
                const double pr = v[p][j] * v[p][k];            // rounded product (-fmad=false: never contracted)
#pragma unroll
                for (int r = 0; r < 6; r++) w[p][r] = fma(tt[6 * q + r], pr, w[p][r]);
            }
            q++;
        }
    }
}

// third-order terms of MATRIX3 (G35): w[p][r] += sum over the triples t = (j,k,l), j <= k <= l, lexicographic, of
// U[r][t] ((v_j v_k) v_l), continuing row r's FMA chain after the second-order terms.  ut = Ut[56][6].
// `zero` (an opaque 0, see matrix_map_uniform) ties every pair product to the accumulator it will feed:
// v_j | (zero & w) is v_j, bit for bit, but cannot be formed before w is: without it ptxas hoists all 77 products of a
// particle to the front of the 1344-DFMA block and spills them.
template <int P>
__device__ __forceinline__ void matrix3_terms(const double* __restrict__ ut, long long zero, const double (&v)[P][6], double (&w)[P][6]) {
    int t = 0;
#pragma unroll
    for (int j = 0; j < 6; j++) {
#pragma unroll
        for (int k = j; k < 6; k++) {
            double pjk[P];
#pragma unroll
            for (int p = 0; p < P; p++) {
                const double vj = __longlong_as_double(__double_as_longlong(v[p][j]) | (zero & __double_as_longlong(w[p][0])));
                pjk[p] = vj * v[p][k];
            }
#pragma unroll
            for (int l = k; l < 6; l++) {
#pragma unroll
                for (int p = 0; p < P; p++) {
                    const double pr = pjk[p] * v[p][l];
#pragma unroll
                    for (int r = 0; r < 6; r++) w[p][r] = fma(ut[6 * t + r], pr, w[p][r]);
                }
                t++;
            }
        }
    }
}

// Zero-pattern specialisation ("may be offered as flagged options and reported separately"): a MATRIX
// whose entries outside the pattern of an uncoupled element are exactly zero,
//     rows x, x': columns x, x', delta;  rows y, y': columns y, y', delta;  row s: all;  row delta: columns s, delta,
// needs 20 of the 36 FMAs.  The kept terms run in the same order as in matrix_map, and a skipped term adds +-0, so
// for finite coordinates the result equals the dense map's (up to the sign of a zero).  c = 28 packed doubles:
// (R00 R01)(R05 C0)(R10 R11)(R15 C1)(R22 R23)(R25 C2)(R32 R33)(R35 C3)(R40 R41)(R42 R43)(R44 R45)(C4 R54)(R55 C5)(- -).
// Coefficients are uniform operands; `zero` makes the row constants vector values (see matrix_map_uniform).
template <int P>
__device__ __forceinline__ void matrix_unc_map_uniform(const double* __restrict__ c, long long zero, const double (&v)[P][6], double (&w)[P][6]) {
#pragma unroll
    for (int h = 0; h < 2; h++) {                                // transverse planes: rows 2h, 2h + 1
#pragma unroll
        for (int rr = 0; rr < 2; rr++) {
            const double* k = c + 8 * h + 4 * rr;                // k[0] k[1] | k[2] = R[.][5], k[3] = C
            const double cv = __longlong_as_double(__double_as_longlong(k[3]) | zero);
#pragma unroll
            for (int p = 0; p < P; p++) {
                double acc = cv;
                acc = fma(k[0], v[p][2 * h], acc);
                acc = fma(k[1], v[p][2 * h + 1], acc);
                acc = fma(k[2], v[p][5], acc);
                w[p][2 * h + rr] = acc;
            }
        }
    }
    const double c4 = __longlong_as_double(__double_as_longlong(c[22]) | zero);
    const double c5 = __longlong_as_double(__double_as_longlong(c[25]) | zero);
#pragma unroll
    for (int p = 0; p < P; p++) {
        double acc = c4;
#pragma unroll
        for (int cc = 0; cc < 6; cc++) acc = fma(c[16 + cc], v[p][cc], acc);
        w[p][4] = acc;
        double a5 = c5;
        a5 = fma(c[23], v[p][4], a5);
        a5 = fma(c[24], v[p][5], a5);
        w[p][5] = a5;
    }
}

// DRIFT, RFKICK and the wake KICK, in place
template <int P, bool EXT = true>
__device__ __forceinline__ void other_map(int ty, const double* __restrict__ c, const ChainCommon& cm, double (&v)[P][6]) {
    if (ty == OP_DRIFT) {                                        // PAPER.md:75-77, G2
        const double L = c[0];
#pragma unroll
        for (int p = 0; p < P; p++) {
            v[p][0] = fma(v[p][1], L, v[p][0]);
            v[p][2] = fma(v[p][3], L, v[p][2]);
            double u = fma(v[p][1], v[p][1], 1.0);
            u = fma(v[p][3], v[p][3], u);
            v[p][4] = fma(L, sqrt(u), v[p][4]);
        }
    } else if (ty == OP_RFKICK) {                                // G8
        const double A = c[0], omega = c[1], phi0 = c[2], inv_bc = c[4];
        const double s_ref = (c[5] != 0.0) ? cm.st->s_ref : c[3];            // G36 (bunch fiducial) / G8 (design)
#pragma unroll
        for (int p = 0; p < P; p++) {
            const double tau = (v[p][4] - s_ref) * inv_bc;
            const double arg = fma(omega, tau, phi0);
            v[p][5] = fma(A, sin(arg), v[p][5]);
        }
    } else if (ty == OP_KICK) {                                  // G14: wake kick of the preceding WAKE
        const double inv_bc = c[0], inv_E = c[1];
        const double t_lo = cm.st->win[0], inv_dt = cm.st->win[2];
        const int nb = cm.nb;
#pragma unroll
        for (int p = 0; p < P; p++) {
            double u0;
            const int b = bin_of(v[p][4], inv_bc, t_lo, inv_dt, nb, &u0);
            if (b < 0) continue;
            double Vt;
            if (!cm.interp || nb < 2) {
                Vt = __ldg(cm.V + b);
            } else {
                const double u = u0 - 0.5;
                double k = floor(u);
                if (k < 0.0) k = 0.0;
                if (k > (double)(nb - 2)) k = (double)(nb - 2);
                double fr = u - k;
                if (fr < 0.0) fr = 0.0;
                if (fr > 1.0) fr = 1.0;
                const int ki = (int)k;
                const double V0 = __ldg(cm.V + ki), V1 = __ldg(cm.V + ki + 1);
                Vt = fma(fr, V1 - V0, V0);
            }
            v[p][5] = fma(-Vt, inv_E, v[p][5]);
        }
    } else if (EXT && ty == OP_TKICK) {                          // G32: x' += Vx(t) / (beta0 p0c), y' likewise
        const double inv_bc = c[0], inv_E = c[1];
        const double t_lo = cm.st->win[0], inv_dt = cm.st->win[2];
        const int nb = cm.t_nb;
#pragma unroll
        for (int p = 0; p < P; p++) {
            double u0;
            const int b = bin_of(v[p][4], inv_bc, t_lo, inv_dt, nb, &u0);
            if (b < 0) continue;
            double vx, vy;
            if (!cm.t_interp || nb < 2) {
                vx = __ldg(cm.Vx + b); vy = __ldg(cm.Vy + b);
            } else {
                const double u = u0 - 0.5;
                double k = floor(u);
                if (k < 0.0) k = 0.0;
                if (k > (double)(nb - 2)) k = (double)(nb - 2);
                double fr = u - k;
                if (fr < 0.0) fr = 0.0;
                if (fr > 1.0) fr = 1.0;
                const int ki = (int)k;
                const double x0 = __ldg(cm.Vx + ki), x1 = __ldg(cm.Vx + ki + 1);
                const double y0 = __ldg(cm.Vy + ki), y1 = __ldg(cm.Vy + ki + 1);
                vx = fma(fr, x1 - x0, x0);
                vy = fma(fr, y1 - y0, y0);
            }
            v[p][1] = fma(vx, inv_E, v[p][1]);
            v[p][3] = fma(vy, inv_E, v[p][3]);
        }
    } else if (EXT && ty == OP_KICK3) {                          // G14 + G32 with a shared bin and interpolation weight:
        const double inv_bc = c[0], inv_E = c[1];                //   the same operations on each coordinate as OP_KICK
        const double t_lo = cm.st->win[0], inv_dt = cm.st->win[2];   // followed by OP_TKICK (neither changes s)
        const int nb = cm.nb;
#pragma unroll
        for (int p = 0; p < P; p++) {
            double u0;
            const int b = bin_of(v[p][4], inv_bc, t_lo, inv_dt, nb, &u0);
            if (b < 0) continue;
            double Vt, vx, vy;
            if (!cm.interp || nb < 2) {
                Vt = __ldg(cm.V + b); vx = __ldg(cm.Vx + b); vy = __ldg(cm.Vy + b);
            } else {
                const double u = u0 - 0.5;
                double k = floor(u);
                if (k < 0.0) k = 0.0;
                if (k > (double)(nb - 2)) k = (double)(nb - 2);
                double fr = u - k;
                if (fr < 0.0) fr = 0.0;
                if (fr > 1.0) fr = 1.0;
                const int ki = (int)k;
                const double V0 = __ldg(cm.V + ki), V1 = __ldg(cm.V + ki + 1);
                const double x0 = __ldg(cm.Vx + ki), x1 = __ldg(cm.Vx + ki + 1);
                const double y0 = __ldg(cm.Vy + ki), y1 = __ldg(cm.Vy + ki + 1);
                Vt = fma(fr, V1 - V0, V0);
                vx = fma(fr, x1 - x0, x0);
                vy = fma(fr, y1 - y0, y0);
            }
            v[p][5] = fma(-Vt, inv_E, v[p][5]);
            v[p][1] = fma(vx, inv_E, v[p][1]);
            v[p][3] = fma(vy, inv_E, v[p][3]);
        }
    }
}

// EXT = false leaves out the second-order map: the HBM-bound short kernels stay at 72 registers (3 blocks per SM); the
// planner picks the EXT = true instantiation when a run holds a MATRIX2.  TK: the transverse wake kick is compiled in
// (chain_kernel always; compact_kernel only with EXT: with the kick in its base form the compaction measured 1.5 %
// slower at 1e8 particles, and a TKICK directly in front of an aperture is rare).
// Without the second-order map the loop over the MAXOPS parameter slots is fully unrolled, so every coefficient has a
// compile-time offset in the constant bank and reaches its DFMA as a uniform-register operand (LDCU + DFMA R, R, UR, R):
// no per-coefficient LDC through the MIO (profiles/r01d: 6 -> 53 DFMA/clk/SM at two particles per thread in a
// register-only loop), no register copy-back after a matrix, no type dispatch at run time (an RFCW cavity's fused run
// -- KICK, TKICK, MATRIX, RFKICK -- ran 443 instructions per particle in the EXT form, 25 % of them moves: 1.99 -> 1.87
// ms per cavity at 1e8 particles).  Only the slots a run uses are ever fetched, so the larger code does not cost
// instruction cache.
template <int MAXOPS, int P, bool EXT, bool TK = false>
__device__ __forceinline__ void apply_ops(const ChainArgs<MAXOPS>& a, double (&v)[P][6]) {
    const int n_ops = a.c.n_ops;
    if constexpr (!EXT) {
#pragma unroll
        for (int op = 0; op < MAXOPS; op++) {
            if (op >= n_ops) break;
            const double* c = a.coef[op];
            const int ty = a.type[op];
            if (ty == OP_MATRIX) {
                double w[P][6];
                matrix_map<P>(c, v, w);
#pragma unroll
                for (int p = 0; p < P; p++)
#pragma unroll
                    for (int r = 0; r < 6; r++) v[p][r] = w[p][r];
            } else {
                other_map<P, TK>(ty, c, a.c, v);
            }
        }
    } else {                                                     // with the second-order code per slot the unrolled form spills
        for (int op = 0; op < n_ops; op++) {
            const double* c = a.coef[op];
            const int ty = a.type[op];
            if (ty == OP_MATRIX || ty == OP_MATRIX2) {
                double w[P][6];
                matrix_map<P>(c, v, w);
                if (ty == OP_MATRIX2) { matrix2_terms<P>(c + 42, v, w); op += 3; }
#pragma unroll
                for (int p = 0; p < P; p++)
#pragma unroll
                    for (int r = 0; r < 6; r++) v[p][r] = w[p][r];
            } else {
                other_map<P, true>(ty, c, a.c, v);
            }
        }
    }
}

__device__ __forceinline__ bool survives(int ap_type, double ax, double ay, double x, double y) {
    if (ap_type == AP_RCOL) return (fabs(x) <= ax) && (fabs(y) <= ay);        // NaN -> false (G17)
    const double xa = x * ax, yb = y * ay;                                    // ECOL: ax, ay hold 1/a, 1/b
    const double r2 = fma(xa, xa, yb * yb);
    return r2 <= 1.0;
}

constexpr unsigned long long kFlagA = 1ull;                  // aggregate available
__device__ __forceinline__ unsigned long long pack_status(unsigned int epoch, unsigned long long flag,
                                                          unsigned long long value) {
    return ((unsigned long long)epoch << 34) | (flag << 32) | value;
}

// ---------------------------------------------------------------------------------------------------
// Moments (a13; G20) as pieces shared by moments_kernel and by the moment EPILOGUE of the fused
// kernels (statistics after an element without a second pass over the particles): shifted one-pass
// sums of d = v - K, a fixed shuffle tree per block, per-block partials combined in block order by the last block
// to finish (the paper's "last block" scheme) -- deterministic for a fixed grid.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void moments_add(double (&acc)[kNMom], const double (&x)[6], const double (&K)[6]) {
    double d[6];
#pragma unroll
    for (int c = 0; c < 6; c++) d[c] = x[c] - K[c];
    int q = 6;
#pragma unroll
    for (int r = 0; r < 6; r++) {
        acc[r] += d[r];
#pragma unroll
        for (int c = r; c < 6; c++) { acc[q] = fma(d[r], d[c], acc[q]); q++; }
    }
}

// every thread of the block calls this once with its sums; n_ptr: where the live count the record reports is found
// (read after every block has finished).  NWARPS warps take part; barrier_id 0 = __syncthreads.
template <int NWARPS, int BAR_ID>
__device__ __forceinline__ void moments_finish(const double (&acc)[kNMom], const double (&K)[6], DevState* st, const long long* n_ptr,
                                               double* partial, double* rec) {
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    __shared__ double s_part[NWARPS][kNMom];
    __shared__ double s_tot[kNMom];
    __shared__ bool s_last;
    auto block_sync = [&]() {
        if constexpr (BAR_ID == 0) __syncthreads();
        else named_barrier<BAR_ID, NWARPS * 32>();
    };
#pragma unroll
    for (int q = 0; q < kNMom; q++) {
        double x = acc[q];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
        if (lane == 0) s_part[wid][q] = x;
    }
    block_sync();
    if (threadIdx.x < kNMom) {
        double x = 0.0;
        for (int w = 0; w < NWARPS; w++) x += s_part[w][threadIdx.x];
        partial[(long long)threadIdx.x * gridDim.x + blockIdx.x] = x;
    }
    __threadfence();
    block_sync();
    if (threadIdx.x == 0) s_last = (atomicAdd(&st->mom_done, 1u) == gridDim.x - 1);
    block_sync();
    if (!s_last) return;
    __threadfence();
    // the last block combines the per-block partials: thread t takes blocks t, t + NT, ... (all 27 loads of a step are
    // independent and in flight together), then the same fixed tree as above
    double tot[kNMom];
#pragma unroll
    for (int q = 0; q < kNMom; q++) tot[q] = 0.0;
    for (int bk = threadIdx.x; bk < (int)gridDim.x; bk += NWARPS * 32) {
        double t[kNMom];
#pragma unroll
        for (int q = 0; q < kNMom; q++) t[q] = __ldcg(partial + (long long)q * gridDim.x + bk);
#pragma unroll
        for (int q = 0; q < kNMom; q++) tot[q] += t[q];
    }
#pragma unroll
    for (int q = 0; q < kNMom; q++) {
        double x = tot[q];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) x += __shfl_xor_sync(0xffffffffu, x, d);
        if (lane == 0) s_part[wid][q] = x;
    }
    block_sync();
    if (threadIdx.x < kNMom) {
        double x = 0.0;
        for (int w = 0; w < NWARPS; w++) x += s_part[w][threadIdx.x];
        s_tot[threadIdx.x] = x;
    }
    block_sync();
    if (threadIdx.x == 0) {
        const long long n = *reinterpret_cast<const volatile long long*>(n_ptr);
        rec[0] = (double)n;
        if (n <= 0) {
            for (int k = 1; k < 43; k++) rec[k] = 0.0;                       // G28
        } else {
            const double inv_n = 1.0 / (double)n;
            double m[6];
            for (int c = 0; c < 6; c++) { m[c] = s_tot[c] * inv_n; rec[1 + c] = K[c] + m[c]; }
            int q = 6;
            for (int r = 0; r < 6; r++)
                for (int c = r; c < 6; c++) {
                    const double val = s_tot[q] * inv_n - m[r] * m[c];
                    rec[7 + 6 * r + c] = val;
                    rec[7 + 6 * c + r] = val;
                    q++;
                }
        }
        st->mom_done = 0;
    }
}

// ---------------------------------------------------------------------------------------------------
// chain_kernel: one launch applies a RUN of consecutive elements to every live particle: each
// coordinate is loaded once (128-bit), carried in registers through all maps and stored once
// (north_star part 1; the paper launches one kernel per element).
//
// Work decomposition: a tile is kBlock * P consecutive particles made of H = P/2 sub-tiles of
// 2 * kBlock; thread t owns particles 2t, 2t+1 of every sub-tile (one 128-bit access per coordinate and
// sub-tile, warp accesses are 512 contiguous bytes).  Only the coordinates the run reads / writes are
// loaded / stored (accessor masks).
// ---------------------------------------------------------------------------------------------------
// The shift K of the moment epilogue: the run's maps applied to particle 0 of the store (every thread computes the
// same K; non-finite components become 0).  It only has to lie inside the distribution (conditioning of the
// one-pass formula: s is an absolute path length), it need not be a survivor.
template <int MAXOPS, bool EXT, bool TK = false>
__device__ __forceinline__ void moment_shift(const ChainArgs<MAXOPS>& a, long long n, double (&K)[6]) {
    double k1[1][6];
#pragma unroll
    for (int cc = 0; cc < 6; cc++) k1[0][cc] = (n > 0) ? __ldg(a.c.src[cc]) : 0.0;
    apply_ops<MAXOPS, 1, EXT, TK>(a, k1);
#pragma unroll
    for (int cc = 0; cc < 6; cc++) K[cc] = (fabs(k1[0][cc]) < INFINITY) ? k1[0][cc] : 0.0;
}

// MOM: the run is followed by a moments record (G26): the 27 shifted sums are accumulated on the mapped particles
// while they are in registers and the record is finished by the last block -- no second pass over the particles.
template <int MAXOPS, int P, bool EXT, bool MOM>
__global__ void __launch_bounds__(kBlock, ((P >= 4 || MOM) ? 2 : 3)) chain_kernel(const __grid_constant__ ChainArgs<MAXOPS> a) {
    pdl_begin();
    constexpr int H = P / 2;                    // sub-tiles per tile
    constexpr int kSub = 2 * kBlock;            // particles per sub-tile
    constexpr int kTileP = kBlock * P;
    const ChainCommon& c = a.c;
    const long long n_all = c.st->n_alive[c.cur];
    const long long n = (c.range_hi >= 0 && c.range_hi < n_all) ? c.range_hi : n_all;       // end of my range
    const long long n_tiles = (n > c.range_lo) ? (n - c.range_lo + kTileP - 1) / kTileP : 0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double mn = INFINITY, mx = -INFINITY;
    account_work(c.st, c.prof_kind, n - c.range_lo, c.bytes_pp, c.flops_pp);
    double K[MOM ? 6 : 1], acc[MOM ? kNMom : 1];
    if constexpr (MOM) {
        moment_shift<MAXOPS, EXT, (ELG_TKICK_BASE != 0)>(a, n, K);
#pragma unroll
        for (int q = 0; q < kNMom; q++) acc[q] = 0.0;
    }

    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long t0 = c.range_lo + tile * kTileP + (long long)threadIdx.x * 2;
        double v[P][6];
#pragma unroll
        for (int h = 0; h < H; h++) {
            const long long i0 = t0 + (long long)h * kSub;
            const bool full = (i0 + 2 <= n);
#pragma unroll
            for (int cc = 0; cc < 6; cc++) {
                v[2 * h][cc] = 0.0; v[2 * h + 1][cc] = 0.0;
                if (c.rmask & (1u << cc)) {
                    if (full) {
                        const double2 t = ld_stream2(c.src[cc] + i0);
                        v[2 * h][cc] = t.x; v[2 * h + 1][cc] = t.y;
                    } else if (i0 < n) {
                        v[2 * h][cc] = ld_stream1(c.src[cc] + i0);
                    }
                }
            }
        }

        apply_ops<MAXOPS, P, EXT, (ELG_TKICK_BASE != 0)>(a, v);

#pragma unroll
        for (int h = 0; h < H; h++) {
            const long long i0 = t0 + (long long)h * kSub;
            const bool full = (i0 + 2 <= n);
#pragma unroll
            for (int cc = 0; cc < 6; cc++) {
                if (c.wmask & (1u << cc)) {
                    if (full) *reinterpret_cast<double2*>(c.dst[cc] + i0) = make_double2(v[2 * h][cc], v[2 * h + 1][cc]);
                    else if (i0 < n) c.dst[cc][i0] = v[2 * h][cc];
                }
            }
            if (c.want_minmax) {
                if (i0 < n) { mn = fmin(mn, v[2 * h][4]); mx = fmax(mx, v[2 * h][4]); }
                if (full) { mn = fmin(mn, v[2 * h + 1][4]); mx = fmax(mx, v[2 * h + 1][4]); }
            }
            if constexpr (MOM) {
                if (i0 < n) moments_add(acc, v[2 * h], K);
                if (full) moments_add(acc, v[2 * h + 1], K);
            }
        }
    }
    if constexpr (MOM) moments_finish<kWarps, 0>(acc, K, c.st, &c.st->n_alive[c.cur], c.mom_partial, c.mom_record);

    if (c.want_minmax) {                                       // exact min/max of s (a8): order-independent
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, d));
            mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        }
        __shared__ double s_mn[kWarps], s_mx[kWarps];
        if (lane == 0) { s_mn[wid] = mn; s_mx[wid] = mx; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < kWarps; w++) { mn = fmin(mn, s_mn[w]); mx = fmax(mx, s_mx[w]); }
            c.mm_partial[2 * blockIdx.x] = mn;
            c.mm_partial[2 * blockIdx.x + 1] = mx;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// chain_long_kernel: long runs of maps (cfg3: 80 MATRIX per launch), the kernel the headline metric spends 97 % of
// its time in.  Bound by the fp64 pipe, and on sm_100 every coefficient that reaches a DFMA through a vector
// register (LDS, LDC, LDG) costs that pipe a write-back slot: with the coefficients in shared memory the bound is
// 36P / (36P + 42) of the DFMA rate for P particles per thread (0.84 at P = 6; round 1 measured 0.80).
// Here the coefficients never touch a vector register: they stay in the kernel-parameter constant bank and reach
// the DFMA as UNIFORM-register operands, loaded by UR-indexed LDCU in the runtime loop over the run's maps
// (LDCU.64 UR, c[0x0][UR+imm]; DFMA R, R, UR, R).  A DFMA takes one uniform operand, so the row constant C[r] is made
// a vector value once per row (matrix_map_uniform); with two uniform operands in the first term ptxas falls back to
// per-thread LDC for everything.  tests/test_abi.py checks the SASS for the uniform form.
// LEVEL 0: MATRIX, DRIFT, RFKICK, KICK; 1: + MATRIX2, TKICK, KICK3; 2: + MATRIX3; 3: level 0 + MATRIX_UNC (flagged option).
// The planner picks the lowest level a run needs; particles per thread, block size and register cap per level below.
// Level 0: 6 particles per thread, one block of 384 threads per SM (168 registers): a register-only loop of 80
// matrices ran at 61.5 DFMA/clk/SM = 96 % of the pipe in a microbenchmark (50.0 with shared-memory coefficients); the
// kernel as it is: fp64 pipe 96.2 % active in ncu (profiles/r02f_final_round2.md, capture G).
// The next tile is prefetched into shared memory with cp.async while the current one is in the pipe, every thread
// copying exactly the 16-byte chunks it will read itself (no block-wide barrier in the tile loop).
// Same arithmetic, in the same order, as chain_kernel.
// ---------------------------------------------------------------------------------------------------
template <int LEVEL> struct LongCfg;
template <> struct LongCfg<0> { static constexpr int NT = ELG_L0_NT, PL = ELG_L0_PL, REGS = ELG_L0_REGS; };
template <> struct LongCfg<1> { static constexpr int NT = ELG_L1_NT, PL = ELG_L1_PL, REGS = ELG_L1_REGS; };
template <> struct LongCfg<2> { static constexpr int NT = ELG_L2_NT, PL = ELG_L2_PL, REGS = ELG_L2_REGS; };
template <> struct LongCfg<3> { static constexpr int NT = 384, PL = 6, REGS = ELG_L3_REGS; };
__host__ __device__ constexpr int long_pl(int level) { return level == 0 ? LongCfg<0>::PL : level == 1 ? LongCfg<1>::PL : level == 2 ? LongCfg<2>::PL : LongCfg<3>::PL; }
template <int LEVEL>
constexpr int chain_long_smem_bytes() { return 6 * LongCfg<LEVEL>::NT * LongCfg<LEVEL>::PL * 8; }

// `zero` is a 0 loaded from the device state (opaque to the compiler, and a per-thread value to it): OR-ing it into the
// bits of C[r] makes C[r] a vector value once per ROW without changing a bit of it, so that every DFMA of the row has
// exactly one uniform operand.
// R rows are formed together, coefficient by coefficient: R x P accumulator chains in flight in SOURCE order.  ptxas
// reschedules, but the order it is given matters: chain after chain (round 1 to mid round 2) ran cfg3 at 0.924 of the
// fp64 peak, one row of P chains at 0.947, two rows at 0.949 (three: 0.943, six: 0.949; profiles/r02d_variants.md); the
// second-order level is best with one row (p4 0.860 against 0.846).  Per chain the FMAs keep their order (G3).
template <int P, int R>
__device__ __forceinline__ void matrix_map_uniform(const double* __restrict__ c, long long zero, const double (&v)[P][6], double (&w)[P][6]) {
    if constexpr (R == 0) {                                      // chain after chain (the order level 3 is fastest with)
#pragma unroll
        for (int r = 0; r < 6; r++) {
            const double cv = __longlong_as_double(__double_as_longlong(c[36 + r]) | zero);
#pragma unroll
            for (int p = 0; p < P; p++) {
                double acc = cv;
#pragma unroll
                for (int cc = 0; cc < 6; cc++) acc = fma(c[6 * r + cc], v[p][cc], acc);
                w[p][r] = acc;
            }
        }
        return;
    }
    constexpr int RR = (R == 0) ? 1 : R;
    static_assert(6 % RR == 0, "rows per group divide 6");
#pragma unroll
    for (int r0 = 0; r0 < 6; r0 += RR) {
        double acc[RR][P];
#pragma unroll
        for (int rr = 0; rr < RR; rr++) {
            const double cv = __longlong_as_double(__double_as_longlong(c[36 + r0 + rr]) | zero);
#pragma unroll
            for (int p = 0; p < P; p++) acc[rr][p] = cv;
        }
#pragma unroll
        for (int cc = 0; cc < 6; cc++)
#pragma unroll
            for (int rr = 0; rr < RR; rr++)
#pragma unroll
                for (int p = 0; p < P; p++) acc[rr][p] = fma(c[6 * (r0 + rr) + cc], v[p][cc], acc[rr][p]);
#pragma unroll
        for (int rr = 0; rr < RR; rr++)
#pragma unroll
            for (int p = 0; p < P; p++) w[p][r0 + rr] = acc[rr][p];
    }
}

template <int MAXOPS, int P, int LEVEL>
__device__ __forceinline__ void apply_ops_uniform(const ChainArgs<MAXOPS>& a, double (&v)[P][6]) {
    const long long zero = a.c.st->zero_bits;                    // 0, but loaded: opaque to the compiler, and a vector value
    constexpr int MMR = (LEVEL == 1) ? ELG_MM_ROWS_L1 : (LEVEL == 3) ? ELG_MM_ROWS_L3 : ELG_MM_ROWS;
    const int n_ops = a.c.n_ops;
    int op = 0;
    while (op < n_ops) {
        const int ty = a.type[op];
        if (ty == OP_MATRIX) {
            const int end = op + a.mat_run[op];                  // [op, end): consecutive MATRIX maps
#pragma unroll 1
            for (; op + 1 < end; op += 2) {                      // pairs: v -> w -> v, no copy-back; nothing else in this loop
                double w[P][6];
                matrix_map_uniform<P, MMR>(a.coef[op], zero, v, w);
                matrix_map_uniform<P, MMR>(a.coef[op + 1], zero, w, v);
            }
            if (op < end) {
                double w[P][6];
                matrix_map_uniform<P, MMR>(a.coef[op], zero, v, w);
#pragma unroll
                for (int p = 0; p < P; p++)
#pragma unroll
                    for (int r = 0; r < 6; r++) v[p][r] = w[p][r];
                op++;
            }
        } else if (LEVEL == 3 && ty == OP_MATRIX_UNC) {
            const int end = op + a.mat_run[op];                  // consecutive MATRIX_UNC maps (host-computed like MATRIX)
#pragma unroll 1
            for (; op + 1 < end; op += 2) {
                double w[P][6];
                matrix_unc_map_uniform<P>(a.coef[op], zero, v, w);
                matrix_unc_map_uniform<P>(a.coef[op + 1], zero, w, v);
            }
            if (op < end) {
                double w[P][6];
                matrix_unc_map_uniform<P>(a.coef[op], zero, v, w);
#pragma unroll
                for (int p = 0; p < P; p++)
#pragma unroll
                    for (int r = 0; r < 6; r++) v[p][r] = w[p][r];
                op++;
            }
        } else if ((LEVEL == 1 || LEVEL == 2) && (ty == OP_MATRIX2 || (LEVEL == 2 && ty == OP_MATRIX3))) {
            double w[P][6];
            matrix_map_uniform<P, MMR>(a.coef[op], zero, v, w);
            matrix2_terms<P>(a.coef[op + 1], v, w);              // slots op + 1 .. op + 3: Tt[21][6]
            if (LEVEL == 2 && ty == OP_MATRIX3) matrix3_terms<P>(a.coef[op + 4], zero, v, w);     // op + 4 .. op + 11: Ut[56][6]
#pragma unroll
            for (int p = 0; p < P; p++)
#pragma unroll
                for (int r = 0; r < 6; r++) v[p][r] = w[p][r];
            op += (ty == OP_MATRIX3) ? 12 : 4;
        } else {
            other_map<P, (LEVEL == 1 || LEVEL == 2)>(ty, a.coef[op], a.c, v);
            op++;
        }
    }
}

template <int MAXOPS, int LEVEL>
__global__ void __maxnreg__(LongCfg<LEVEL>::REGS) chain_long_kernel(const __grid_constant__ ChainArgs<MAXOPS> a) {
    pdl_begin();
    constexpr int PL = LongCfg<LEVEL>::PL;
    constexpr int NT = LongCfg<LEVEL>::NT, NW = NT / 32;
    constexpr int kTileL = NT * PL;
    constexpr int H = PL / 2;
    constexpr int kSub = 2 * NT;
    static_assert(PL % 2 == 0, "128-bit accesses: particles per thread come in pairs");
    extern __shared__ __align__(16) double s_tile0[];            // [6][H][kSub]: thread t owns doubles 2t, 2t+1 of each row
    const ChainCommon& c = a.c;
    const long long n_all = c.st->n_alive[c.cur];
    const long long n = (c.range_hi >= 0 && c.range_hi < n_all) ? c.range_hi : n_all;       // end of my range
    const long long n_tiles = (n > c.range_lo) ? (n - c.range_lo + kTileL - 1) / kTileL : 0;
    __shared__ double s_mn[NT], s_mx[NT];                        // running min / max of s per thread: not in registers,
    if (c.want_minmax) { s_mn[threadIdx.x] = INFINITY; s_mx[threadIdx.x] = -INFINITY; }     // the map loop needs them all
    account_work(c.st, c.prof_kind, n - c.range_lo, c.bytes_pp, c.flops_pp);

    auto prefetch = [&](long long tile) {
        const long long t0 = c.range_lo + tile * kTileL + (long long)threadIdx.x * 2;
#pragma unroll
        for (int h = 0; h < H; h++) {
            const long long i0 = t0 + (long long)h * kSub;
            const long long left = n - i0;
            const int bytes = left >= 2 ? 16 : (left == 1 ? 8 : 0);          // zero-fill beyond the live prefix
            const long long is = left >= 1 ? i0 : 0;
#pragma unroll
            for (int cc = 0; cc < 6; cc++)
                if (c.rmask & (1u << cc))
                    cp_async16(s_tile0 + (cc * H + h) * kSub + threadIdx.x * 2, c.src[cc] + is, bytes);
        }
    };

    long long tile = blockIdx.x;
    if (tile < n_tiles) prefetch(tile);
    while (tile < n_tiles) {
        double v[PL][6];
        cp_async_wait_all();
#pragma unroll
        for (int h = 0; h < H; h++)
#pragma unroll
            for (int cc = 0; cc < 6; cc++) {
                double2 t = make_double2(0.0, 0.0);
                if (c.rmask & (1u << cc)) t = *reinterpret_cast<const double2*>(s_tile0 + (cc * H + h) * kSub + threadIdx.x * 2);
                v[2 * h][cc] = t.x; v[2 * h + 1][cc] = t.y;
            }
        const long long next = tile + gridDim.x;
        if (next < n_tiles) prefetch(next);                      // own slots only: already in registers

        apply_ops_uniform<MAXOPS, PL, LEVEL>(a, v);

        const long long t0 = c.range_lo + tile * kTileL + (long long)threadIdx.x * 2;
#pragma unroll
        for (int h = 0; h < H; h++) {
            const long long i0 = t0 + (long long)h * kSub;
            const bool full = (i0 + 2 <= n);
#pragma unroll
            for (int cc = 0; cc < 6; cc++) {
                if (c.wmask & (1u << cc)) {
                    if (full) *reinterpret_cast<double2*>(c.dst[cc] + i0) = make_double2(v[2 * h][cc], v[2 * h + 1][cc]);
                    else if (i0 < n) c.dst[cc][i0] = v[2 * h][cc];
                }
            }
            if (c.want_minmax) {
                double mn = s_mn[threadIdx.x], mx = s_mx[threadIdx.x];
                if (i0 < n) { mn = fmin(mn, v[2 * h][4]); mx = fmax(mx, v[2 * h][4]); }
                if (full) { mn = fmin(mn, v[2 * h + 1][4]); mx = fmax(mx, v[2 * h + 1][4]); }
                s_mn[threadIdx.x] = mn; s_mx[threadIdx.x] = mx;
            }
        }
        tile = next;
    }

    if (c.want_minmax) {                                         // exact min/max of s (a8)
        const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
        double mn = s_mn[threadIdx.x], mx = s_mx[threadIdx.x];
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, d));
            mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        }
        __syncthreads();
        if (lane == 0) { s_mn[wid] = mn; s_mx[wid] = mx; }
        __syncthreads();
        if (threadIdx.x == 0) {
            for (int w = 1; w < NW; w++) { mn = fmin(mn, s_mn[w]); mx = fmax(mx, s_mx[w]); }
            c.mm_partial[2 * blockIdx.x] = mn;
            c.mm_partial[2 * blockIdx.x + 1] = mx;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// compact_kernel: a run of maps that ends in an aperture (a6) followed by the stable stream compaction
// (a7; north_star part 2): survivors are written out of place in their original order, lost particles
// are appended to the lost log in position order.  Single pass over HBM (56 B read + 56 B written per
// live particle).  The grid is persistent and launched cooperatively (every block resident); tiles of
// TILE = NT x PP particles are dealt round-robin, iteration i of block b works on tile b + i x gridDim.
//
// A tile lives in one stage of a shared-memory ring of S stages from its arrival to the moment its survivors
// leave for global memory; registers hold a particle only while it is mapped.
//   producer warp (one lane): waits until a stage has been released (mbarrier, NT arrivals) and refills it with
//       seven 1-D bulk copies (TMA unit, cp.async.bulk, completion counted in bytes on the stage's "full"
//       mbarrier): the load stream runs F = S - D - 1 tiles ahead of the compute warps, uses no registers, no
//       L1 and seven instructions per tile, and never waits for the scan;
//   compute warps, iteration i:
//   (a) the status words needed for the base of the tile of iteration i - D are requested;
//   (b) wait for tile i (mbarrier try_wait on its stage);
//   (c) every thread loads its PP particles (slots t + q NT), applies the run's maps (coefficients as uniform
//       operands from the parameter bank) and evaluates the aperture;
//   (d) ranks: one __ballot_sync + __popc per sub-tile (the flags are single bits; the lanes of a warp hold
//       consecutive particles), warp totals to shared memory; the polled status words are summed per warp here
//       too, so that ONE named barrier per tile serves both;
//   (e) the tile's survivor count is published at once as a 64-bit status word (epoch | flag | count);
//   (f) the mapped particles are scattered back INTO THE SAME STAGE in compacted order: survivors to slots
//       [0, total), lost ones to [total, valid);
//   (g) the tile of iteration i - D has its base by now (own inclusive prefix one tile earlier + the
//       gridDim - 1 aggregates in between, no chained look-back; D = 2 iterations of slack keep the chain
//       "publish <- poll <- publish" of the blocks from ever stalling: D = 1 costs 25 %); thread t copies
//       slots t + m NT of that stage to dst[base + slot]: dense 256-byte warp stores; slots past the survivors
//       go to the lost log at n_lost + (index - survivors before); then the stage is released.
// Measured variants (tile sizes, ring depths, per-thread cp.async instead of bulk copies, round 1's
// register-held tile of round 1): profiles/r02_compact.md.
// ---------------------------------------------------------------------------------------------------
#ifndef ELG_C2_NT
#define ELG_C2_NT 256
#endif
#ifndef ELG_C2_PP
#define ELG_C2_PP 2
#endif
#ifndef ELG_C2_S
#define ELG_C2_S 4
#endif
#ifndef ELG_C2_D
#define ELG_C2_D 2
#endif
#ifndef ELG_C2_BLOCKS
#define ELG_C2_BLOCKS 2
#endif
constexpr int kC2NT = ELG_C2_NT;                        // compute threads per block
constexpr int kC2PP = ELG_C2_PP;                        // particles per thread and tile
constexpr int kC2S = ELG_C2_S;                          // ring stages
constexpr int kC2D = ELG_C2_D;                          // a tile's base is resolved D iterations after its count
constexpr int kC2Tile = kC2NT * kC2PP;
constexpr int kC2Threads = kC2NT + 32;                  // + the producer warp
constexpr int kPoll = 3;                                // status words per thread and tile
constexpr int kCompactMaxGrid = kPoll * kC2NT + 1;
constexpr int kStatusTile = 256;                        // tile_status is sized for tiles of at least this many particles
constexpr int compact_smem_bytes() { return kC2S * 7 * kC2Tile * 8; }

template <int MAXOPS, bool EXT, bool MOM>
__global__ void __launch_bounds__(kC2Threads, (MOM ? 1 : ELG_C2_BLOCKS)) compact_kernel(const __grid_constant__ ChainArgs<MAXOPS> a) {
    pdl_begin();
    constexpr int NT = kC2NT, PP = kC2PP, S = kC2S, D = kC2D, TILE = kC2Tile, NW = NT / 32;
    static_assert(D >= 1 && S - D - 1 >= 0, "ring: S = D + F + 1");
    static_assert(kC2Tile >= kStatusTile && kC2Tile % 2 == 0, "tile_status capacity; 16-byte bulk copies");
    const ChainCommon& c = a.c;
    const long long n = c.st->n_alive[c.cur];
    const long long n_tiles = (n + TILE - 1) / TILE;
    const long long lost_base = c.st->n_lost[c.cur];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    const unsigned int lt_mask = (1u << lane) - 1u;
    double mn = INFINITY, mx = -INFINITY;
    account_work(c.st, c.prof_kind, n, c.bytes_pp, c.flops_pp);

    extern __shared__ __align__(16) double c2_ring[];           // [S][7][TILE]; row 6 holds the IDs (bit patterns)
    __shared__ int s_wtot[2][PP][NW];                            // per iteration parity, sub-tile, warp: survivors
    __shared__ unsigned int s_part[2][NW];                       // per iteration parity, warp: polled aggregates
    __shared__ unsigned long long s_full[S], s_empty[S];         // mbarriers: tile landed / stage released by all readers

    const long long G = gridDim.x;
    const long long n_it = (n_tiles > blockIdx.x) ? (n_tiles - blockIdx.x + G - 1) / G : 0;     // my tiles

    if (threadIdx.x == 0) {
        for (int k = 0; k < S; k++) { mbar_init(&s_full[k], 1); mbar_init(&s_empty[k], NT); }
        mbar_fence_init();
    }
    __syncthreads();
    if (wid == NW) {                                             // producer warp: one lane feeds the ring
        if (lane == 0) {
            for (long long it = 0; it < n_it; it++) {
                const int stg = (int)(it % S);
                const long long use = it / S;
                if (use > 0) mbar_wait(&s_empty[stg], (unsigned int)((use - 1) & 1));
                const long long tile = blockIdx.x + it * G;
                const long long left = n - tile * TILE;
                // whole 16-byte units; an odd tail reads one element past n, inside the array's 256-byte padding
                const unsigned int bytes = (unsigned int)(((left < TILE ? left : TILE) + 1) / 2) * 16u;
                double* stage = c2_ring + (size_t)stg * 7 * TILE;
                mbar_expect_tx(&s_full[stg], 7u * bytes);
#pragma unroll
                for (int cc = 0; cc < 6; cc++) bulk_g2s(stage + cc * TILE, c.src[cc] + tile * TILE, bytes, &s_full[stg]);
                bulk_g2s(stage + 6 * TILE, c.id_src + tile * TILE, bytes, &s_full[stg]);
            }
        }
        return;
    }

    int tot_hist[D];                                             // survivor counts of the last D counted tiles
#pragma unroll
    for (int d = 0; d < D; d++) tot_hist[d] = 0;
    long long my_incl = 0;                                       // inclusive survivor prefix at my last resolved tile
    double K[MOM ? 6 : 1], acc[MOM ? kNMom : 1];                 // moment epilogue over the survivors (G26)
    if constexpr (MOM) {
        moment_shift<MAXOPS, EXT>(a, n, K);
#pragma unroll
        for (int q = 0; q < kNMom; q++) acc[q] = 0.0;
    }

    for (long long it = 0; it < n_it + D; it++) {
        const int par = (int)(it & 1);
        const long long r = it - D;                              // the iteration whose tile is resolved and stored now
        const bool cur_valid = it < n_it, res_valid = r >= 0 && r < n_it;
        const long long rtile = blockIdx.x + r * G;              // (only meaningful when res_valid)

        // (a) aggregates between my previous tile and tile r, published at least D - 1 iterations ago
        unsigned long long stt[kPoll];
        const long long first = (r > 0) ? rtile - G + 1 : 0;     // tiles [first, rtile)
#pragma unroll
        for (int j = 0; j < kPoll; j++) {
            const long long w = first + threadIdx.x + j * NT;
            stt[j] = (res_valid && w < rtile) ? ld_relaxed(c.tile_status + w) : pack_status(c.epoch, kFlagA, 0);
        }

        int total = 0;
        bool ok[PP], surv[PP];
        double v[PP][6];
        long long id[PP];
        unsigned int bal[PP];
        double* stage = c2_ring + (size_t)(it % S) * 7 * TILE;
        if (cur_valid) {
            const long long tile = blockIdx.x + it * G;
            mbar_wait(&s_full[it % S], (unsigned int)((it / S) & 1));    // (b)
#pragma unroll
            for (int q = 0; q < PP; q++) {                       // (c)
                const int slot = threadIdx.x + q * NT;
                ok[q] = tile * TILE + slot < n;                  // slots past n hold stale bytes: never used
#pragma unroll
                for (int cc = 0; cc < 6; cc++) v[q][cc] = stage[cc * TILE + slot];
                id[q] = __double_as_longlong(stage[6 * TILE + slot]);
            }
            apply_ops<MAXOPS, PP, EXT>(a, v);
#pragma unroll
            for (int q = 0; q < PP; q++) {                       // (d)
                surv[q] = ok[q] && survives(c.ap_type, c.ap_x, c.ap_y, v[q][0], v[q][2]);
                bal[q] = __ballot_sync(0xffffffffu, surv[q]);
                if (lane == 0) s_wtot[par][q][wid] = __popc(bal[q]);
            }
        }
        if (res_valid) {                                         // the polled aggregates, summed per warp
            unsigned int part = 0;
#pragma unroll
            for (int j = 0; j < kPoll; j++) {
                const long long w = first + threadIdx.x + j * NT;
                if (w < rtile) {
                    while ((unsigned int)(stt[j] >> 34) != c.epoch || ((stt[j] >> 32) & 3ull) == 0) stt[j] = ld_relaxed(c.tile_status + w);
                    part += (unsigned int)(stt[j] & 0xffffffffull);
                }
            }
            part = __reduce_add_sync(0xffffffffu, part);
            if (lane == 0) s_part[par][wid] = part;
        }
        named_barrier<1, NT>();                                  // the one barrier per tile (compute warps): stage read by all, totals visible

        if (cur_valid) {
            const long long tile = blockIdx.x + it * G;
            int before[PP];                                      // survivors before my warp's part of sub-tile q
#pragma unroll
            for (int q = 0; q < PP; q++) {
                int sub = 0, mine = 0;
#pragma unroll
                for (int w = 0; w < NW; w++) {
                    const int x = s_wtot[par][q][w];
                    if (w < wid) mine += x;
                    sub += x;
                }
                before[q] = total + mine;
                total += sub;
            }
            if (threadIdx.x == 0 && tile + 1 < n_tiles)          // (e)
                st_relaxed(c.tile_status + tile, pack_status(c.epoch, kFlagA, (unsigned long long)total));
#pragma unroll
            for (int q = 0; q < PP; q++) {                       // (f) compacted order inside the stage
                const int slot = threadIdx.x + q * NT;
                const int rank = before[q] + __popc(bal[q] & lt_mask);
                const int pos = surv[q] ? rank : total + (slot - rank);
                if (ok[q]) {
#pragma unroll
                    for (int cc = 0; cc < 6; cc++) stage[cc * TILE + pos] = v[q][cc];
                    stage[6 * TILE + pos] = __longlong_as_double(id[q]);
                    if (c.want_minmax && surv[q]) { mn = fmin(mn, v[q][4]); mx = fmax(mx, v[q][4]); }
                    if constexpr (MOM) { if (surv[q]) moments_add(acc, v[q], K); }
                }
            }
        }

        if (res_valid) {                                         // (g)
            long long base = my_incl;
#pragma unroll
            for (int w = 0; w < NW; w++) base += s_part[par][w];
            const int rtotal = tot_hist[D - 1];
            my_incl = base + rtotal;
            if (rtile == n_tiles - 1 && threadIdx.x == 0) {      // the last tile knows the totals
                c.st->n_alive[c.cur ^ 1] = my_incl;
                c.st->n_lost[c.cur ^ 1] = lost_base + (n - my_incl);
            }
            const long long left = n - rtile * TILE;
            const int rvalid = left < TILE ? (int)left : TILE;
            const long long lost0 = lost_base + (rtile * TILE - base);       // lost before the tile = index - survivors before
            const double* rs = c2_ring + (size_t)(r % S) * 7 * TILE;
#pragma unroll
            for (int m = 0; m < PP; m++) {
                const int slot = threadIdx.x + m * NT;
                if (slot < rtotal) {
                    const long long d = base + slot;
#pragma unroll
                    for (int cc = 0; cc < 6; cc++) c.dst[cc][d] = rs[cc * TILE + slot];
                    c.id_dst[d] = __double_as_longlong(rs[6 * TILE + slot]);
                } else if (slot < rvalid) {
                    const long long lpos = lost0 + (slot - rtotal);
                    if (lpos < c.lost_cap) {
                        c.lost_id[lpos] = __double_as_longlong(rs[6 * TILE + slot]);
                        c.lost_te[lpos] = c.te_code;
#pragma unroll
                        for (int cc = 0; cc < 6; cc++) c.lost_v[cc * c.lost_cap + lpos] = rs[cc * TILE + slot];
                    }
                }
            }
            fence_proxy_async();                                 // my generic-proxy accesses before the next bulk write
            mbar_arrive(&s_empty[r % S]);                        // stage released (NT arrivals complete the phase)
        }
#pragma unroll
        for (int d = D - 1; d > 0; d--) tot_hist[d] = tot_hist[d - 1];
        tot_hist[0] = total;
    }

    if (c.want_minmax) {                                         // exact min/max of s over the survivors (a8)
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, d));
            mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        }
        __shared__ double s_mn[NW], s_mx[NW];
        if (lane == 0) { s_mn[wid] = mn; s_mx[wid] = mx; }
        named_barrier<1, NT>();
        if (threadIdx.x == 0) {
            for (int w = 1; w < NW; w++) { mn = fmin(mn, s_mn[w]); mx = fmax(mx, s_mx[w]); }
            c.mm_partial[2 * blockIdx.x] = mn;
            c.mm_partial[2 * blockIdx.x + 1] = mx;
        }
    }
    if (n_tiles == 0 && blockIdx.x == 0 && threadIdx.x == 0) {   // nothing alive: carry the counts over
        c.st->n_alive[c.cur ^ 1] = 0;
        c.st->n_lost[c.cur ^ 1] = lost_base;
    }
    // the survivor count of the record was written above by the block that resolved the last tile, before its arrival
    if constexpr (MOM) moments_finish<NW, 1>(acc, K, c.st, &c.st->n_alive[c.cur ^ 1], c.mom_partial, c.mom_record);
}

// ---------------------------------------------------------------------------------------------------
// chain_ring_kernel: the HBM-bound short run (at most two matrices, basic maps) with the LOAD side of compact_kernel:
// a producer warp keeps a shared-memory ring of S tiles full with 1-D bulk copies (TMA unit, one per coordinate the run
// reads, completion counted in bytes on the stage's mbarrier), the compute warps take a tile out of its stage into
// registers, release the stage at once, apply the run's maps and store with 128-bit st.global.  The load stream no
// longer stops while a warp computes or stores (chain_kernel holds its in-flight loads in registers).  Same arithmetic,
// same order, as chain_kernel; tiles are dealt round-robin to a persistent grid.  Measured at 1e8 particles
// (profiles/r02d_variants.md): DRIFT + MATRIX 1.626 -> 1.584 ms (6.06 TB/s) with 2 stages and 3 blocks per SM; 3 - 5
// stages at 2 blocks per SM are slower, and so is the moment epilogue on this structure (one block of 8 compute warps
// per SM: 1.15 -> 1.27 ms), which therefore stays with chain_kernel.
// ---------------------------------------------------------------------------------------------------
#ifndef ELG_CR_BLOCKS
#define ELG_CR_BLOCKS 3
#endif
#ifndef ELG_CR_S
#define ELG_CR_S 2
#endif
constexpr int kCrNT = 256;                              // compute threads per block (+ one producer warp)
constexpr int kCrTile = 2 * kCrNT;                      // thread t owns particles 2t, 2t + 1 of the tile
constexpr int kCrS = ELG_CR_S;                          // ring stages
constexpr int kCrThreads = kCrNT + 32;
constexpr int chain_ring_smem_bytes() { return kCrS * 6 * kCrTile * 8; }

template <int MAXOPS>
__global__ void __launch_bounds__(kCrThreads, ELG_CR_BLOCKS) chain_ring_kernel(const __grid_constant__ ChainArgs<MAXOPS> a) {
    pdl_begin();
    constexpr int NT = kCrNT, TILE = kCrTile, S = kCrS, NW = NT / 32;
    const ChainCommon& c = a.c;
    const long long n_all = c.st->n_alive[c.cur];
    const long long n = (c.range_hi >= 0 && c.range_hi < n_all) ? c.range_hi : n_all;       // end of my range
    const long long n_tiles = (n > c.range_lo) ? (n - c.range_lo + TILE - 1) / TILE : 0;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    account_work(c.st, c.prof_kind, n - c.range_lo, c.bytes_pp, c.flops_pp);

    extern __shared__ __align__(16) double cr_ring[];            // [S][6][TILE]
    __shared__ unsigned long long s_full[S], s_empty[S];         // mbarriers: tile landed / stage read by all
    const long long G = gridDim.x;
    const long long n_it = (n_tiles > blockIdx.x) ? (n_tiles - blockIdx.x + G - 1) / G : 0;  // my tiles

    if (threadIdx.x == 0) {
        for (int k = 0; k < S; k++) { mbar_init(&s_full[k], 1); mbar_init(&s_empty[k], NT); }
        mbar_fence_init();
    }
    __syncthreads();
    if (wid == NW) {                                             // producer warp: one lane feeds the ring
        if (lane == 0) {
            const unsigned int n_rd = (unsigned int)__popc(c.rmask & 0x3Fu);
            for (long long it = 0; it < n_it; it++) {
                const int stg = (int)(it % S);
                const long long use = it / S;
                if (use > 0) mbar_wait(&s_empty[stg], (unsigned int)((use - 1) & 1));
                const long long i0 = c.range_lo + (blockIdx.x + it * G) * TILE;
                const long long left = n - i0;
                // whole 16-byte units; an odd tail reads one element past n, inside the array's 256-byte padding
                const unsigned int bytes = (unsigned int)(((left < TILE ? left : TILE) + 1) / 2) * 16u;
                double* stage = cr_ring + (size_t)stg * 6 * TILE;
                mbar_expect_tx(&s_full[stg], n_rd * bytes);
#pragma unroll
                for (int cc = 0; cc < 6; cc++)
                    if (c.rmask & (1u << cc)) bulk_g2s(stage + cc * TILE, c.src[cc] + i0, bytes, &s_full[stg]);
            }
        }
        return;
    }

    double mn = INFINITY, mx = -INFINITY;

    for (long long it = 0; it < n_it; it++) {
        const int stg = (int)(it % S);
        const long long i0 = c.range_lo + (blockIdx.x + it * G) * TILE + (long long)threadIdx.x * 2;
        const double* stage = cr_ring + (size_t)stg * 6 * TILE + threadIdx.x * 2;
        mbar_wait(&s_full[stg], (unsigned int)((it / S) & 1));
        double v[2][6];
#pragma unroll
        for (int cc = 0; cc < 6; cc++) {
            double2 t = make_double2(0.0, 0.0);
            if (c.rmask & (1u << cc)) t = *reinterpret_cast<const double2*>(stage + cc * TILE);
            v[0][cc] = t.x; v[1][cc] = t.y;
        }
        fence_proxy_async();                                     // my generic-proxy reads before the next bulk write
        mbar_arrive(&s_empty[stg]);                              // stage released (NT arrivals complete the phase)
        const bool full = (i0 + 2 <= n), one = (i0 < n);         // slots past n hold stale bytes: mapped, never used

        apply_ops<MAXOPS, 2, false, (ELG_TKICK_BASE != 0)>(a, v);

#pragma unroll
        for (int cc = 0; cc < 6; cc++) {
            if (c.wmask & (1u << cc)) {
                if (full) *reinterpret_cast<double2*>(c.dst[cc] + i0) = make_double2(v[0][cc], v[1][cc]);
                else if (one) c.dst[cc][i0] = v[0][cc];
            }
        }
        if (c.want_minmax) {
            if (one) { mn = fmin(mn, v[0][4]); mx = fmax(mx, v[0][4]); }
            if (full) { mn = fmin(mn, v[1][4]); mx = fmax(mx, v[1][4]); }
        }
    }

    if (c.want_minmax) {                                         // exact min/max of s (a8): order-independent
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, d));
            mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
        }
        __shared__ double s_mn[NW], s_mx[NW];
        if (lane == 0) { s_mn[wid] = mn; s_mx[wid] = mx; }
        named_barrier<1, NT>();
        if (threadIdx.x == 0) {
            for (int w = 1; w < NW; w++) { mn = fmin(mn, s_mn[w]); mx = fmax(mx, s_mx[w]); }
            c.mm_partial[2 * blockIdx.x] = mn;
            c.mm_partial[2 * blockIdx.x + 1] = mx;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// window_kernel (a8 -> G10): reduce the per-block min/max partials (exact in any order), derive the
// histogram window with the same fp64 operations as the definition, the occupied bin range used for
// shared-memory privatisation, and zero the counts (every block zeroes a slice, block 0 does the rest).
// ---------------------------------------------------------------------------------------------------
struct WindowArgs {
    DevState* st;
    int cur;
    const double* mm_partial;
    int n_partial;
    int mode;            // ELG_WIN_*
    int nb;
    double t_lo_rel, dt_in, t_design, inv_bc;
    unsigned int* counts;
    long long* dacc;     // TRWAKE: 4 * nb fixed-point dipole accumulators to zero as well (or NULL)
};

__global__ void __launch_bounds__(kBlock) window_kernel(const WindowArgs a) {
    pdl_begin();
    for (int i = blockIdx.x * kBlock + threadIdx.x; i < a.nb; i += gridDim.x * kBlock) a.counts[i] = 0u;   // all blocks
    if (a.dacc)
        for (int i = blockIdx.x * kBlock + threadIdx.x; i < 4 * a.nb; i += gridDim.x * kBlock) a.dacc[i] = 0;
    if (blockIdx.x != 0) return;                                 // block 0 derives the window
    __shared__ double s_mn[kWarps], s_mx[kWarps];
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    double mn = INFINITY, mx = -INFINITY;
    for (int i = threadIdx.x; i < a.n_partial; i += kBlock) {
        mn = fmin(mn, a.mm_partial[2 * i]);
        mx = fmax(mx, a.mm_partial[2 * i + 1]);
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        mn = fmin(mn, __shfl_xor_sync(0xffffffffu, mn, d));
        mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, d));
    }
    if (lane == 0) { s_mn[wid] = mn; s_mx[wid] = mx; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kWarps; w++) { mn = fmin(mn, s_mn[w]); mx = fmax(mx, s_mx[w]); }
        const long long n = a.st->n_alive[a.cur];
        if (n == 0) { mn = 0.0; mx = 0.0; }                                  // G28
        double t_lo, dt;
        const double t_min = mn * a.inv_bc, t_max = mx * a.inv_bc;
        if (a.mode == 0) {                                                   // EXPLICIT
            t_lo = a.t_design + a.t_lo_rel;
            dt = a.dt_in;
        } else if (a.mode == 1) {                                            // AUTO_MINMAX
            dt = (t_max - t_min) / (double)(a.nb - 1);
            if (!(dt > 0.0)) dt = 1e-15;
            t_lo = t_min - 0.5 * dt;
        } else {                                                             // AUTO_TABLE
            dt = a.dt_in;
            const double tc = 0.5 * (t_min + t_max);
            t_lo = tc - (0.5 * (double)a.nb) * dt;
        }
        const double inv_dt = 1.0 / dt;
        a.st->win[0] = t_lo; a.st->win[1] = dt; a.st->win[2] = inv_dt; a.st->win[3] = 0.0;
        a.st->smin = mn; a.st->smax = mx;
        // the bin function is monotone in s, so every particle falls in [bin(smin), bin(smax)]
        long long lo = (long long)floor(fmax(fmin((mn * a.inv_bc - t_lo) * inv_dt, 4.0e9), -4.0e9));
        long long hi = (long long)floor(fmax(fmin((mx * a.inv_bc - t_lo) * inv_dt, 4.0e9), -4.0e9));
        if (lo < 0) lo = 0;
        if (hi > a.nb - 1) hi = a.nb - 1;
        if (n == 0 || !(mn <= mx)) { lo = 0; hi = -1; }
        a.st->bin_lo = lo; a.st->bin_hi = hi;
    }
}

// ---------------------------------------------------------------------------------------------------
// hist_kernel (a9): threads increment shared-memory bins atomically; several private
// sub-histograms per block (one per warp when they fit) cut contention; sub-histograms are combined
// with integer global atomics (exact, order-independent).  Only the occupied bin range is privatised,
// so nb = 65536 (256 KB) still fits; bins outside the first kHistSmemBins of the range fall back to
// global atomics.  Persistent grid, 4 x 128-bit loads of s per thread and iteration.
// ---------------------------------------------------------------------------------------------------
struct HistArgs {
    const double* s;
    DevState* st;
    int prof_kind;
    int cur;
    long long n_fixed;     // >= 0: use this n and the explicit window below (test hook); < 0: device state
    double inv_bc, t_lo, inv_dt;
    int nb;
    int aggregate;         // 1: warp-aggregate equal bins with match.any before the shared atomic (hist_kernel<true>)
    int smem_bins;         // bins of dynamic shared memory this launch was given (<= kHistSmemBins)
    unsigned int* counts;
};

template <bool AGG>
__global__ void __launch_bounds__(kBlock, 6) hist_kernel(const HistArgs a) {
    pdl_begin();
    extern __shared__ unsigned int sh[];
    long long n, blo, bhi;
    double t_lo, inv_dt;
    if (a.n_fixed >= 0) { n = a.n_fixed; blo = 0; bhi = a.nb - 1; t_lo = a.t_lo; inv_dt = a.inv_dt; }
    else { n = a.st->n_alive[a.cur]; blo = a.st->bin_lo; bhi = a.st->bin_hi; t_lo = a.st->win[0]; inv_dt = a.st->win[2]; }
    if (a.st) account_work(a.st, a.prof_kind, n, 8u, 4u);
    long long span = bhi - blo + 1;
    if (span < 1) span = 1;
    const int S = (int)(span < a.smem_bins ? span : a.smem_bins);
    int R = a.smem_bins / S;
    if (R > kWarps) R = kWarps;
    const int wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    unsigned int* mine = sh + (wid % R) * S;
    for (int i = threadIdx.x; i < R * S; i += kBlock) sh[i] = 0u;
    __syncthreads();
    const int lo32 = (int)blo;                                   // 0 <= bin_lo <= nb - 1 < 2^24

    constexpr int kPer = 8;                                      // 4 x 128-bit loads in flight per thread
    const long long stride = (long long)gridDim.x * kBlock * kPer;
    // warp-uniform trip count (the aggregated path uses full-mask warp votes)
    for (long long w0 = ((long long)blockIdx.x * kBlock + (threadIdx.x & ~31)) * kPer; w0 < n; w0 += stride) {
        // lane l owns particles w0 + 2l + 64k + {0, 1}, k < 4: every load is a 512-byte warp access
        const long long i0 = w0 + (long long)lane * 2;
        double sv[kPer];
        bool have[kPer];
        if (w0 + 32 * kPer <= n) {                               // the whole warp chunk is live: no per-load tests
#pragma unroll
            for (int k = 0; k < kPer / 2; k++) {
                const double2 t = ld_stream2(a.s + i0 + 64 * k);
                sv[2 * k] = t.x; sv[2 * k + 1] = t.y; have[2 * k] = true; have[2 * k + 1] = true;
            }
        } else {
#pragma unroll
            for (int k = 0; k < kPer / 2; k++) {
                const long long i = i0 + 64 * k;
                have[2 * k] = i < n; have[2 * k + 1] = i + 1 < n;
                sv[2 * k] = 0.0; sv[2 * k + 1] = 0.0;
                if (have[2 * k + 1]) { const double2 t = ld_stream2(a.s + i); sv[2 * k] = t.x; sv[2 * k + 1] = t.y; }
                else if (have[2 * k]) sv[2 * k] = ld_stream1(a.s + i);
            }
        }
        if constexpr (!AGG) {
            // branch-free common path: one predicated shared-memory reduction per particle (the kernel is bound by
            // instruction issue, not by memory: 8 bytes per particle); bins outside the privatised range are rare and
            // take the global atomics in a second pass over the registers
            const unsigned int mine32 = smem_u32(mine);
            int bb[kPer];
            bool fallback = false;
#pragma unroll
            for (int p = 0; p < kPer; p++) {
                double u;
                const int b = bin_of(sv[p], a.inv_bc, t_lo, inv_dt, a.nb, &u);
                bb[p] = have[p] ? b : -1;
                const unsigned int rel = (unsigned int)(bb[p] - lo32);       // (wraps past S when b < bin_lo or b = -1)
                const bool in_s = bb[p] >= 0 && rel < (unsigned int)S;
                asm volatile("{\n.reg .pred q;\nsetp.ne.s32 q, %1, 0;\n@q red.shared.add.u32 [%0], 1;\n}" ::"r"(mine32 + rel * 4u), "r"((int)in_s) : "memory");
                fallback |= bb[p] >= 0 && !in_s;
            }
            if (fallback) {
#pragma unroll
                for (int p = 0; p < kPer; p++)
                    if (bb[p] >= 0 && (unsigned int)(bb[p] - lo32) >= (unsigned int)S) atomicAdd(a.counts + bb[p], 1u);
            }
            continue;
        }
#pragma unroll
        for (int p = 0; p < kPer; p++) {
            double u;
            const int b = have[p] ? bin_of(sv[p], a.inv_bc, t_lo, inv_dt, a.nb, &u) : -1;
            const unsigned int rel = (unsigned int)(b - lo32);   // b < bin_lo cannot happen (monotone bin function); if it
                                                                 // did, rel wraps past S and the global path takes it
            if constexpr (AGG) {
                const unsigned int act = __ballot_sync(0xffffffffu, b >= 0);   // loop trip count is warp-uniform
                if (b >= 0) {
                    const unsigned int peers = __match_any_sync(act, b);
                    if ((int)(__ffs(peers) - 1) == lane) {
                        if (rel < (unsigned int)S) atomicAdd(mine + rel, (unsigned int)__popc(peers));
                        else atomicAdd(a.counts + b, (unsigned int)__popc(peers));
                    }
                }
            } else if (b >= 0) {
                if (rel < (unsigned int)S) atomicAdd(mine + rel, 1u);
                else atomicAdd(a.counts + b, 1u);
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < S; i += kBlock) {
        unsigned int tot = 0;
        for (int r = 0; r < R; r++) tot += sh[r * S + i];
        if (tot) atomicAdd(a.counts + blo + i, tot);
    }
}

// ---------------------------------------------------------------------------------------------------
// dipole_hist_kernel (TRWAKE, G32-G33): bin counts and per-bin dipole sums of x and y.  A sum of doubles
// accumulated with atomics would depend on the order of arrival; here every coordinate is split exactly into
// two integers (hi = rint(x 2^36), lo = rint((x - hi 2^-36) 2^64)) which are summed with 64-bit
// INTEGER arithmetic: exact to 2^-64 m per particle, order-independent, run-to-run reproducible.
// Shared-memory privatisation of the occupied bin range as in hist_kernel, 36 bytes per bin, laid out as NINE
// PLANES of 32-bit words (count | low and high words of the four 64-bit sums): the word of bin b in a plane sits in
// bank b mod 32, so the 32 lanes of an atomic spread over all banks (round 1 kept the four 64-bit sums of a bin side by
// side: every atomic of a warp fell into 4 of the 32 banks, 85 % of the shared-memory wavefront peak, 0.74 ms per
// 1e8 particles; profiles/r02c_dipole.md).  The split point 2^36 (round 1: 2^32) leaves both integers of a
// millimetre-sized offset below 2^28, so the low word of a sum rarely wraps and an add is ONE native 32-bit atomic
// (the carry into the high word follows in 1-3 % of the adds): 5.1 shared atomics per particle instead of 9.
// ---------------------------------------------------------------------------------------------------
constexpr int kDipoleSmemBins = 1792;                   // 1792 x 36 B = 63 KB: the most bins a block privatises
#ifndef ELG_DIP_PER
#define ELG_DIP_PER 4
#endif
#ifndef ELG_DIP_BLOCKS
#define ELG_DIP_BLOCKS 4
#endif
constexpr int kDipolePer = ELG_DIP_PER;                 // particles per thread and iteration: 6 x 128-bit loads in flight
constexpr int kFixDipole = 36;                          // split point of the dipole sums: |sum of x over a bin| < 2^27 m
constexpr int kFixFiducial = 32;                        // split point of the fiducial sum (no shared atomics there: keep the
                                                        // larger range, |sum of s - s_design| < 2^31 m)
constexpr double kFixLo = 18446744073709551616.0;       // 2^64

struct DipoleArgs {
    const double* s;
    const double* x;
    const double* y;
    DevState* st;
    int prof_kind;
    int cur;
    double inv_bc;
    int nb;
    int smem_bins;                 // bins of dynamic shared memory this launch was given (<= kDipoleSmemBins)
    unsigned int* counts;
    unsigned long long* dacc;      // [nb][4]: x hi, x lo, y hi, y lo
};

template <int BITS>
__device__ __forceinline__ bool fixed_split(double x, long long* hi, long long* lo) {
    constexpr double kHi = (double)(1ull << BITS);
    if (!(fabs(x) < 1048576.0)) return false;
    const double h = rint(x * kHi);
    const double r = x - h * (1.0 / kHi);                        // exact
    *hi = (long long)h;
    *lo = (long long)rint(r * kFixLo);                           // (rounding by adding 1.5 x 2^52 as in bin_of was
    return true;                                                 //  measured here too: slower, the fp64 pipe is the busier one)
}
template <int BITS>
__device__ __forceinline__ double fixed_join(long long H, long long L) {
    constexpr double kHi = (double)(1ull << BITS);
    return fma((double)H, 1.0 / kHi, (double)L * (1.0 / kFixLo));
}

// 64-bit integer adds in shared memory from native 32-bit atomics (a 64-bit shared atomicAdd compiles to a
// compare-and-swap spin loop): add the low word, carry into the high word when the low word wrapped.  Addition
// modulo 2^64 commutes, so the result does not depend on the interleaving.  A small negative value has high word
// 0xffffffff and nearly always produces a carry: hi + carry = 0, one atomic as well.  The four low-word atomics of a
// particle are issued back to back (independent), the rare high-word ones follow.
__device__ __forceinline__ void smem_add64x4(unsigned int* planes, int S, int rel, const unsigned long long (&v)[4]) {
    unsigned int old[4];
#pragma unroll
    for (int k = 0; k < 4; k++) old[k] = atomicAdd(planes + (1 + 2 * k) * S + rel, (unsigned int)v[k]);
#pragma unroll
    for (int k = 0; k < 4; k++) {
        const unsigned int lo = (unsigned int)v[k], hi = (unsigned int)(v[k] >> 32);
        const unsigned int up = hi + ((old[k] + lo < old[k]) ? 1u : 0u);
        if (up) atomicAdd(planes + (2 + 2 * k) * S + rel, up);
    }
}

__global__ void __launch_bounds__(kBlock, ELG_DIP_BLOCKS) dipole_hist_kernel(const DipoleArgs a) {
    pdl_begin();
    extern __shared__ __align__(16) unsigned int sh_dip[];       // [9][S]
    const long long n = a.st->n_alive[a.cur];
    const long long blo = a.st->bin_lo, bhi = a.st->bin_hi;
    const double t_lo = a.st->win[0], inv_dt = a.st->win[2];
    account_work(a.st, a.prof_kind, n, 24u, 12u);
    long long span = bhi - blo + 1;
    if (span < 1) span = 1;
    const int S = (int)(span < a.smem_bins ? span : a.smem_bins);
    for (int i = threadIdx.x; i < 9 * S; i += kBlock) sh_dip[i] = 0u;
    __syncthreads();
    unsigned int* const sc = sh_dip;
    constexpr int kPer = kDipolePer;
    const long long stride = (long long)gridDim.x * kBlock * kPer;
    // lane l of a warp owns particles w0 + 2l + 64k + {0, 1}, k < kPer / 2: every load is a 512-byte warp access
    for (long long w0 = ((long long)blockIdx.x * kBlock + (threadIdx.x & ~31)) * kPer; w0 < n; w0 += stride) {
        const long long i0 = w0 + (long long)(threadIdx.x & 31) * 2;
        double sv[kPer], xv[kPer], yv[kPer];
        bool have[kPer];
#pragma unroll
        for (int k = 0; k < kPer / 2; k++) {
            const long long i = i0 + 64 * k;
            have[2 * k] = i < n; have[2 * k + 1] = i + 1 < n;
            sv[2 * k] = 0.0; sv[2 * k + 1] = 0.0; xv[2 * k] = 0.0; xv[2 * k + 1] = 0.0; yv[2 * k] = 0.0; yv[2 * k + 1] = 0.0;
            if (have[2 * k + 1]) {
                const double2 ts = ld_stream2(a.s + i), tx = ld_stream2(a.x + i), ty = ld_stream2(a.y + i);
                sv[2 * k] = ts.x; sv[2 * k + 1] = ts.y; xv[2 * k] = tx.x; xv[2 * k + 1] = tx.y; yv[2 * k] = ty.x; yv[2 * k + 1] = ty.y;
            } else if (have[2 * k]) {
                sv[2 * k] = ld_stream1(a.s + i); xv[2 * k] = ld_stream1(a.x + i); yv[2 * k] = ld_stream1(a.y + i);
            }
        }
#pragma unroll
        for (int p = 0; p < kPer; p++) {
            if (!have[p]) continue;
            double u;
            const int b = bin_of(sv[p], a.inv_bc, t_lo, inv_dt, a.nb, &u);
            if (b < 0) continue;
            long long xh, xl, yh, yl;
            const bool ok = fixed_split<kFixDipole>(xv[p], &xh, &xl) & fixed_split<kFixDipole>(yv[p], &yh, &yl);
            const long long rel = (long long)b - blo;
            if (rel < S) {
                const int r = (int)rel;
                atomicAdd(sc + r, 1u);
                if (ok) {
                    const unsigned long long v4[4] = {(unsigned long long)xh, (unsigned long long)xl, (unsigned long long)yh, (unsigned long long)yl};
                    smem_add64x4(sh_dip, S, r, v4);
                }
            } else {
                atomicAdd(a.counts + b, 1u);
                if (ok) {
                    atomicAdd(a.dacc + 4 * (long long)b + 0, (unsigned long long)xh); atomicAdd(a.dacc + 4 * (long long)b + 1, (unsigned long long)xl);
                    atomicAdd(a.dacc + 4 * (long long)b + 2, (unsigned long long)yh); atomicAdd(a.dacc + 4 * (long long)b + 3, (unsigned long long)yl);
                }
            }
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < S; i += kBlock) {
        const unsigned int cnt = sc[i];
        if (cnt) {
            atomicAdd(a.counts + blo + i, cnt);
#pragma unroll
            for (int k = 0; k < 4; k++) {
                const unsigned long long v = (unsigned long long)sh_dip[(1 + 2 * k) * S + i] | ((unsigned long long)sh_dip[(2 + 2 * k) * S + i] << 32);
                if (v) atomicAdd(a.dacc + 4 * (blo + i) + k, v);
            }
        }
    }
}

// D = fma((double)H, 2^-36, (double)L 2^-64) (G33), Dx then Dy
__global__ void __launch_bounds__(kBlock) dipole_finalize_kernel(const unsigned long long* dacc, int nb, double* D) {
    pdl_begin();
    const int k = blockIdx.x * kBlock + threadIdx.x;
    if (k >= nb) return;
    const long long xh = (long long)dacc[4 * k + 0], xl = (long long)dacc[4 * k + 1];
    const long long yh = (long long)dacc[4 * k + 2], yl = (long long)dacc[4 * k + 3];
    D[k] = fixed_join<kFixDipole>(xh, xl);
    D[nb + k] = fixed_join<kFixDipole>(yh, yl);
}

// ---------------------------------------------------------------------------------------------------
// fiducial_kernel (G36; the reduction of simple_rf_cavity): s_ref = s_design + (exact fixed-point
// sum of s_i - s_design) / n.  64-bit integer sums per thread, shuffle tree, one global integer atomic per block;
// the last block to finish converts, publishes s_ref in the device state and re-arms the accumulators.
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock) fiducial_kernel(const double* s, DevState* st, int cur, double s_design) {
    pdl_begin();
    const long long n = st->n_alive[cur];
    long long H = 0, L = 0;
    const long long stride = (long long)gridDim.x * kBlock * 2;
    for (long long i0 = ((long long)blockIdx.x * kBlock + threadIdx.x) * 2; i0 < n; i0 += stride) {
        double a, b = 0.0;
        const bool two = i0 + 2 <= n;
        if (two) { const double2 t = ld_stream2(s + i0); a = t.x; b = t.y; }
        else a = ld_stream1(s + i0);
        long long h, l;
        if (fixed_split<kFixFiducial>(a - s_design, &h, &l)) { H += h; L += l; }
        if (two && fixed_split<kFixFiducial>(b - s_design, &h, &l)) { H += h; L += l; }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
        H += __shfl_xor_sync(0xffffffffu, H, d);
        L += __shfl_xor_sync(0xffffffffu, L, d);
    }
    __shared__ long long s_h[kWarps], s_l[kWarps];
    __shared__ bool s_last;
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) { s_h[wid] = H; s_l[wid] = L; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < kWarps; w++) { H += s_h[w]; L += s_l[w]; }
        atomicAdd(&st->fid_acc[0], (unsigned long long)H);
        atomicAdd(&st->fid_acc[1], (unsigned long long)L);
        __threadfence();
        s_last = (atomicAdd(&st->fid_done, 1u) == gridDim.x - 1);
        if (s_last) {
            __threadfence();
            const long long Ht = (long long)atomicAdd(&st->fid_acc[0], 0ull), Lt = (long long)atomicAdd(&st->fid_acc[1], 0ull);
            const double sum = fixed_join<kFixFiducial>(Ht, Lt);
            st->s_ref = (n > 0) ? s_design + sum / (double)n : s_design;
            st->fid_acc[0] = 0ull; st->fid_acc[1] = 0ull; st->fid_done = 0;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// wake_samples_kernel (a10; G11, G12): W_k = W(k dt), k < nb, in V/C.
// ---------------------------------------------------------------------------------------------------
struct WakeArgs {
    const DevState* st;    // dt from win[1] unless dt_fixed > 0
    double dt_fixed;
    int kind;              // ELG_WAKE_*
    int nb;
    double kloss, alpha, wbar, ratio;     // resonator constants, computed once on the host at load time
    const double* table;
    long long n_table;
    double dt_table;
    double* W;
};

__global__ void __launch_bounds__(kBlock) wake_samples_kernel(const WakeArgs a) {
    pdl_begin();
    const int k = blockIdx.x * kBlock + threadIdx.x;
    if (k >= a.nb) return;
    const double dt = (a.dt_fixed > 0.0) ? a.dt_fixed : a.st->win[1];
    double w;
    if (a.kind == 2) {                                                       // transverse resonator (G34)
        if (k == 0) w = 0.0;
        else {
            const double tau = (double)k * dt;
            w = a.kloss * exp(-a.alpha * tau) * sin(a.wbar * tau);          // kloss holds (w_r Rs / Q)(w_r / wbar)
        }
    } else if (a.kind == 0) {
        if (k == 0) w = a.kloss;                                             // beam-loading theorem (G11)
        else {
            const double tau = (double)k * dt;
            w = 2.0 * a.kloss * exp(-a.alpha * tau) * (cos(a.wbar * tau) - a.ratio * sin(a.wbar * tau));
        }
    } else {
        if (dt == a.dt_table) {
            w = (k < a.n_table) ? a.table[k] : 0.0;
        } else {
            const double pos = ((double)k * dt) / a.dt_table;
            const double fl = floor(pos);
            if (!(fl >= 0.0) || fl > (double)(a.n_table - 1)) w = 0.0;
            else {
                const long long j = (long long)fl;
                const double fr = pos - fl;
                if (j == a.n_table - 1) w = (fr == 0.0) ? a.table[j] : 0.0;
                else w = a.table[j] + fr * (a.table[j + 1] - a.table[j]);
            }
        }
    }
    a.W[k] = w;
}

// ---------------------------------------------------------------------------------------------------
// conv_kernel (a11, G13): V_i = q sum_{j<=i} counts_j W_{i-j}.  The paper's version
// accumulates partial results with fp64 atomicAdd (order non-deterministic); here one warp owns one
// output: lanes take j = j0 + lane (step 32) in ascending order and a fixed butterfly combines them,
// so the result is run-to-run deterministic.  Empty bins outside the occupied range are skipped
// (they contribute exact zeros).
// ---------------------------------------------------------------------------------------------------
template <class T>
struct ConvArgs {
    const T* counts;       // weights: bin counts (WAKE) or dipole sums (TRWAKE)
    const double* W;
    const DevState* st;    // occupied range; NULL: whole range
    int nb;
    double q;
    double* V;
};

template <class T>
__global__ void __launch_bounds__(kBlock) conv_kernel(const ConvArgs<T> a) {
    pdl_begin();
    const int lane = threadIdx.x & 31;
    const int i = blockIdx.x * kWarps + (threadIdx.x >> 5);
    if (i >= a.nb) return;
    long long jlo = 0, jhi = i;
    if (a.st) {
        if (a.st->bin_lo > jlo) jlo = a.st->bin_lo;
        if (a.st->bin_hi < jhi) jhi = a.st->bin_hi;
    }
    double acc = 0.0;
    for (long long j = jlo + lane; j <= jhi; j += 32) acc = fma((double)a.counts[j], a.W[i - j], acc);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (lane == 0) a.V[i] = a.q * acc;
}

// ---------------------------------------------------------------------------------------------------
// conv_rec_kernel (G37): the resonator wake voltage in O(nb) instead of the O(nb^2) convolution.
// W_k = Re[B z^k] with z = exp((-alpha + i wbar) dt), so S_{i+1} = z (S_i + c_i), V_i = q (c_i k_loss + Re[B S_i]).
// One block: every thread runs the recurrence over its own contiguous segment from S = 0, thread 0 chains the
// 256 segment ends with z^L, then every thread repeats its segment from its carry-in and writes V.  Fixed
// decomposition, hence deterministic; it differs from the sequential recurrence only by rounding (<< 1e-10).
// ---------------------------------------------------------------------------------------------------
struct ConvRecArgs {
    const unsigned int* counts;
    const DevState* st;    // dt = win[1]
    int nb;
    double q;
    double kloss, alpha, wbar, ratio;
    double* V;
};

__global__ void __launch_bounds__(kBlock) conv_rec_kernel(const ConvRecArgs a) {
    pdl_begin();
    __shared__ double s_er[kBlock], s_ei[kBlock];
    const double dt = a.st->win[1];
    const int L = (a.nb + kBlock - 1) / kBlock;
    const int lo = threadIdx.x * L, hi = (lo + L < a.nb) ? lo + L : a.nb;
    const double damp = exp(-a.alpha * dt);
    const double zr = damp * cos(a.wbar * dt), zi = damp * sin(a.wbar * dt);
    double Sr = 0.0, Si = 0.0;
    for (int i = lo; i < hi; i++) {
        const double tr = Sr + (double)a.counts[i], ti = Si;
        Sr = fma(zr, tr, -(zi * ti));
        Si = fma(zr, ti, zi * tr);
    }
    // a segment shorter than L (the tail) still has to advance its end state by the missing steps for the chaining
    for (int i = (hi > lo ? hi : lo); i < lo + L; i++) {
        const double tr = Sr, ti = Si;
        Sr = fma(zr, tr, -(zi * ti));
        Si = fma(zr, ti, zi * tr);
    }
    s_er[threadIdx.x] = Sr; s_ei[threadIdx.x] = Si;
    __syncthreads();
    if (threadIdx.x == 0) {                                      // carry-in of segment t: C_{t+1} = z^L C_t + E_t
        const double dL = exp(-a.alpha * dt * (double)L);
        const double pr = dL * cos(a.wbar * dt * (double)L), pi = dL * sin(a.wbar * dt * (double)L);
        double Cr = 0.0, Ci = 0.0;
        for (int t = 0; t < kBlock; t++) {
            const double er = s_er[t], ei = s_ei[t];
            s_er[t] = Cr; s_ei[t] = Ci;
            const double nr = fma(pr, Cr, -(pi * Ci)) + er;
            const double ni = fma(pr, Ci, pi * Cr) + ei;
            Cr = nr; Ci = ni;
        }
    }
    __syncthreads();
    Sr = s_er[threadIdx.x]; Si = s_ei[threadIdx.x];
    const double Br = 2.0 * a.kloss, Bi = 2.0 * a.kloss * a.ratio;
    for (int i = lo; i < hi; i++) {
        const double c = (double)a.counts[i];
        a.V[i] = a.q * fma(c, a.kloss, fma(Br, Sr, -(Bi * Si)));
        const double tr = Sr + c, ti = Si;
        Sr = fma(zr, tr, -(zi * ti));
        Si = fma(zr, ti, zi * tr);
    }
}

// ---------------------------------------------------------------------------------------------------
// moments_kernel (a13; G20): n, centroid and 6x6 central second moments in one
// pass over the six coordinate arrays.  s is an absolute path length, so raw second
// moments would cancel catastrophically; sums are taken of (v - K) with K = coordinates of the first
// live particle (a shift inside the distribution), which makes the one-pass formula well conditioned.
// Deterministic: fixed grid, fixed per-thread order, shuffle tree, partials combined in block order by
// the last block to finish (the paper's "last block" scheme).
// ---------------------------------------------------------------------------------------------------
struct MomArgs {
    const double* src[6];
    DevState* st;
    int cur;
    int prof_kind;
    double* partial;       // [kNMom][gridDim.x]
    double* record;        // 43 doubles: n, C[6], Sigma[36]
};

__global__ void __launch_bounds__(kBlock) moments_kernel(const MomArgs a) {
    pdl_begin();
    const long long n = a.st->n_alive[a.cur];
    account_work(a.st, a.prof_kind, n, 48u, 60u);
    double K[6];
#pragma unroll
    for (int c = 0; c < 6; c++) K[c] = (n > 0) ? __ldg(a.src[c]) : 0.0;
    double acc[kNMom];
#pragma unroll
    for (int q = 0; q < kNMom; q++) acc[q] = 0.0;

    const long long stride = (long long)gridDim.x * kTile;
    for (long long i0 = (long long)blockIdx.x * kTile + (long long)threadIdx.x * kP; i0 < n; i0 += stride) {
        double x[kP][6];
        const bool full = (i0 + kP <= n);
#pragma unroll
        for (int c = 0; c < 6; c++) {
            if (full) {
                const double2 t = ld_stream2(a.src[c] + i0);
                x[0][c] = t.x; x[1][c] = t.y;
            } else {
                x[0][c] = ld_stream1(a.src[c] + i0); x[1][c] = 0.0;
            }
        }
        moments_add(acc, x[0], K);
        if (full) moments_add(acc, x[1], K);
    }
    moments_finish<kWarps, 0>(acc, K, a.st, &a.st->n_alive[a.cur], a.partial, a.record);
}

// ---------------------------------------------------------------------------------------------------
// fp64_peak_kernel: the denominator of the fp64 roofline, measured instead of derived: eight independent DFMA chains
// per thread, nothing else in the loop.  Operand form DFMA R, R, R, c[..] (two vector registers + one constant-bank
// operand): the fastest form on sm_100 (63.5 DFMA/clk/SM; three vector registers or two uniform operands give 58.5)
// and the form of the long-run kernel's own DFMAs (two registers + one uniform).  elg_dbg_fp64_peak times it.
// ---------------------------------------------------------------------------------------------------
constexpr int kPeakIlp = 8, kPeakUnroll = 16;
__global__ void __launch_bounds__(kBlock) fp64_peak_kernel(double* out, long long iters, double b, double c) {
    double a[kPeakIlp];
#pragma unroll
    for (int i = 0; i < kPeakIlp; i++) a[i] = 1e-3 * (threadIdx.x + i);
    const double bb = b + 1e-9 * threadIdx.x;                                    // a per-thread value: vector operand
    for (long long it = 0; it < iters; it++) {
#pragma unroll
        for (int r = 0; r < kPeakUnroll; r++)
#pragma unroll
            for (int i = 0; i < kPeakIlp; i++) a[i] = fma(a[i], bb, c);         // c: kernel parameter = constant-bank operand
    }
    double s = 0.0;
#pragma unroll
    for (int i = 0; i < kPeakIlp; i++) s += a[i];
    if (s == 123.456) out[threadIdx.x] = s;                                     // never true: keeps the chains alive
}

// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(kBlock) iota_kernel(long long* id, long long n) {
    pdl_begin();
    const long long stride = (long long)gridDim.x * kBlock;
    for (long long i = (long long)blockIdx.x * kBlock + threadIdx.x; i < n; i += stride) id[i] = i;
}

__global__ void init_state_kernel(DevState* st, long long n0) {
    pdl_begin();
    st->n_alive[0] = n0; st->n_alive[1] = n0;
    st->n_lost[0] = 0; st->n_lost[1] = 0;
    st->win[0] = 0.0; st->win[1] = 1.0; st->win[2] = 1.0; st->win[3] = 0.0;
    st->smin = 0.0; st->smax = 0.0;
    st->bin_lo = 0; st->bin_hi = -1;
    st->tile_counter = 0; st->done_counter = 0; st->mom_done = 0; st->fid_done = 0;
    st->fid_acc[0] = 0ull; st->fid_acc[1] = 0ull; st->s_ref = 0.0;
    st->zero_bits = 0;                                           // (work[] is not touched: it belongs to elg_profile_read)
}

}  // namespace elg
