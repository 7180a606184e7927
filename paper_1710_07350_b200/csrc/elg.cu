// elg.cu -- C ABI of libelg (include/elg.h): host-side planning and kernel launches.
// Build: nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -fmad=false -shared -Xcompiler -fPIC
// The host code holds no particle arithmetic: it cuts the beamline into fused runs, fills kernel
// parameter blocks and launches the kernels of elg_kernels.cuh.  There is no CPU fallback.
#include "../../include/elg.h"
#include "elg_kernels.cuh"

#include <atomic>
#include <map>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <new>
#include <cstdlib>
#include <string>
#include <utility>
#include <vector>

using namespace elg;

namespace {

thread_local std::string g_err;
std::atomic<long long> g_launches{0};

int32_t fail(int32_t code, const std::string& msg) { g_err = msg; return code; }

#define ELG_CK(call)                                                                           \
    do {                                                                                       \
        cudaError_t e_ = (call);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(ELG_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_));        \
    } while (0)

// Every kernel is launched with the programmatic-stream-serialization attribute (programmatic dependent launch): the
// kernels' first statement is pdl_begin() = griddepcontrol.wait (elg_kernels.cuh), so the ordering is that of the stream
// and only the launch latency between dependent kernels overlaps.  ELG_PDL=0 launches without it.
// ELG_CHAIN_RING=0: short runs through chain_kernel (loads held in registers) instead of chain_ring_kernel
bool ring_enabled() {
    static const bool on = [] { const char* e = std::getenv("ELG_CHAIN_RING"); return !(e && std::atoi(e) == 0); }();
    return on;
}
bool pdl_enabled() {
    static const bool on = [] { const char* e = std::getenv("ELG_PDL"); return !(e && std::atoi(e) == 0); }();
    return on;
}
template <class... KArgs, class... Args>
void launch_k(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t stream, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = pdl_enabled() ? 1 : 0;
    cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);      // errors surface in the caller's cudaGetLastError
}

constexpr double kCLight = 299792458.0;                 // m/s
constexpr double kTwoPi = 6.283185307179586476925286766559;
constexpr int kMaxOpsSmall = 8;
constexpr int kMaxOpsLarge = 80;                        // 80 x 42 x 8 B = 26.9 KB of kernel parameters
constexpr int kMatricesForP4 = 3;                       // runs with >= 3 MATRIX maps use 4 particles per thread
constexpr int kMatricesForLong = 5;                     // runs with >= 5 use the long-run kernel
constexpr int kMaxGrid = 4096;
constexpr int kMmPartials = 16384;                      // min/max partial pairs: blocks x chunks of a pipelined upload
constexpr long long kRecCap = 2048;                     // device ring of moment records
constexpr int kNbDefault = 65536;

inline long long align_up(long long x, long long a) { return (x + a - 1) / a * a; }

struct HostOp {
    uint8_t type;
    double coef[42];
    double dense[42];      // OP_MATRIX_UNC only: the dense coefficients, in case the run cannot use the pattern kernel
};

struct ResConst { double kloss, alpha, wbar, ratio; };

}  // namespace

struct elg_beamline {
    std::vector<elg_element> e;
    std::vector<std::vector<double>> R, C, table, T, U;
    std::vector<ResConst> res;
    std::vector<double> s_design;
    double length = 0.0;
    int32_t ring = 0;
    int32_t nb_max = 0;
    long long table_total = 0;
    std::vector<long long> table_off;                   // offset of element k's table in the device copy
    unsigned long long serial = 0;
};

struct elg_bunch {
    long long n0 = 0, stride = 0, lost_cap = 0, work_bytes = 0;
    char* d_soa = nullptr;
    char* d_work = nullptr;
    cudaStream_t stream = nullptr;
    double p0c = 0, mc2 = 0, charge = 0, beta0 = 0, inv_bc = 0, inv_E = 0, q_macro = 0;
    // workspace carve-up
    DevState* st = nullptr;
    char* soaB = nullptr;
    unsigned long long* tile_status = nullptr;
    double* mm_partial = nullptr;
    double* mom_partial = nullptr;
    double* records = nullptr;
    unsigned int* counts = nullptr;
    double* W = nullptr;
    double* V = nullptr;
    unsigned long long* dacc = nullptr;
    double* D = nullptr;
    double* Vt = nullptr;
    double* table = nullptr;
    long long nb_cap = 0, table_cap = 0;
    long long* lost_id = nullptr;
    long long* lost_te = nullptr;
    double* lost_v = nullptr;
    // dynamic state mirrored on the host without any device read
    int cur_buf = 0;                                    // 0: d_soa, 1: workspace copy
    int cur_slot = 0;
    unsigned int epoch = 0;
    long long turn = 0;
    unsigned long long table_serial = 0;
    long long rec_count = 0;                            // records in the device ring
    // launch geometry
    int sms = 0;
    std::map<int, int> hist_grids;                      // hist_kernel grid per shared-memory size
    std::map<const void*, int> grids;                   // persistent grid size per chain kernel instantiation
    int force_p = 0;                                    // ELG_CHAIN_P = 2 | 4 overrides the planner's choice
    int grid_mom = 0;
    std::map<int, int> dipole_grids;                    // dipole_hist_kernel grid per shared-memory size
    int hist_aggregate = 0;
    // pipelined upload (elg_upload_and_track): the library's own copy stream and one event per chunk
    cudaStream_t copy_stream = nullptr;
    cudaEvent_t entry_ev = nullptr;
    std::vector<cudaEvent_t> chunk_ev;
    // optional per-kernel event timing (elg_profile_*)
    bool prof_on = false;
    struct ProfRec { int kind; cudaEvent_t t0, t1; };
    std::vector<ProfRec> prof_recs;
    std::vector<cudaEvent_t> prof_pool;
    long long prof_launches[ELG_K_COUNT] = {0};
    double prof_ms[ELG_K_COUNT] = {0};

    cudaEvent_t prof_event() {
        cudaEvent_t e = nullptr;
        if (!prof_pool.empty()) { e = prof_pool.back(); prof_pool.pop_back(); }
        else if (cudaEventCreate(&e) != cudaSuccess) e = nullptr;
        return e;
    }
    // drain finished records into the per-kind sums (the caller has synchronised the stream)
    void prof_drain() {
        for (ProfRec& r : prof_recs) {
            float ms = 0.f;
            if (r.t0 && r.t1 && cudaEventElapsedTime(&ms, r.t0, r.t1) == cudaSuccess) {
                prof_launches[r.kind]++;
                prof_ms[r.kind] += (double)ms;
            }
            if (r.t0) prof_pool.push_back(r.t0);
            if (r.t1) prof_pool.push_back(r.t1);
        }
        prof_recs.clear();
    }

    double* coord(int buf, int c) const { return reinterpret_cast<double*>((buf ? soaB : d_soa) + (long long)c * stride * 8); }
    long long* ids(int buf) const { return reinterpret_cast<long long*>((buf ? soaB : d_soa) + 6LL * stride * 8); }
};

namespace {

unsigned long long g_bl_serial = 0;

// brackets one kernel launch with CUDA events when profiling is on
struct ProfScope {
    elg_bunch* b;
    int idx = -1;
    ProfScope(elg_bunch* b_, int kind) : b(b_) {
        if (!b || !b->prof_on) return;
        elg_bunch::ProfRec r{kind, b->prof_event(), b->prof_event()};
        if (r.t0) cudaEventRecord(r.t0, b->stream);
        b->prof_recs.push_back(r);
        idx = (int)b->prof_recs.size() - 1;
    }
    ~ProfScope() {
        if (idx >= 0 && b->prof_recs[idx].t1) cudaEventRecord(b->prof_recs[idx].t1, b->stream);
    }
};

// ------------------------------------------------------------------------------------- workspace
struct WorkLayout {
    long long off_state, off_soaB, off_status, off_mm, off_mom, off_rec, off_counts, off_W, off_V, off_dacc, off_D, off_Vt, off_table,
        off_lost_id, off_lost_te, off_lost_v, total;
};

WorkLayout layout(long long n0, long long nb_cap, long long table_cap, long long lost_cap) {
    WorkLayout L{};
    const long long stride = elg_soa_stride(n0);
    long long o = 0;
    L.off_state = o; o = align_up(o + (long long)sizeof(DevState), 256);
    L.off_soaB = o; o = align_up(o + 7 * stride * 8, 256);
    L.off_status = o; o = align_up(o + (stride / kStatusTile + 2) * 8, 256);
    L.off_mm = o; o = align_up(o + 2LL * kMmPartials * 8, 256);
    L.off_mom = o; o = align_up(o + (long long)kNMom * kMaxGrid * 8, 256);
    L.off_rec = o; o = align_up(o + (kRecCap + 1) * 43 * 8, 256);   // + 1: elg_moments' own slot
    L.off_counts = o; o = align_up(o + nb_cap * 4, 256);
    L.off_W = o; o = align_up(o + nb_cap * 8, 256);
    L.off_V = o; o = align_up(o + nb_cap * 8, 256);
    L.off_dacc = o; o = align_up(o + 4 * nb_cap * 8, 256);         // TRWAKE: fixed-point dipole accumulators
    L.off_D = o; o = align_up(o + 2 * nb_cap * 8, 256);            //         Dx, Dy
    L.off_Vt = o; o = align_up(o + 2 * nb_cap * 8, 256);           //         Vx, Vy
    L.off_table = o; o = align_up(o + table_cap * 8, 256);
    L.off_lost_id = o; o = align_up(o + lost_cap * 8, 256);
    L.off_lost_te = o; o = align_up(o + lost_cap * 8, 256);
    L.off_lost_v = o; o = align_up(o + 6 * lost_cap * 8, 256);
    L.total = o;
    return L;
}

void caps_for(const elg_beamline* bl, long long* nb_cap, long long* table_cap) {
    *nb_cap = bl ? (bl->nb_max > 2 ? bl->nb_max : 2) : kNbDefault;
    *table_cap = bl ? (bl->table_total > 1 ? bl->table_total : 1) : kNbDefault;
}

template <class K>
int32_t grid_for(K kernel, int sms, int smem, int threads, int* out) {
    int occ = 0;
    ELG_CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem));
    if (occ < 1) return fail(ELG_ECUDA, "kernel does not fit on an SM");
    long long g = (long long)occ * sms;
    if (g > kMaxGrid) g = kMaxGrid / sms * sms;
    *out = (int)g;
    return ELG_OK;
}

int32_t device_sms(int* sms) {
    int dev = 0;
    ELG_CK(cudaGetDevice(&dev));
    ELG_CK(cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev));
    return ELG_OK;
}

int32_t long_setup_once() {
    static bool done = false;
    if (!done) {
        ELG_CK(cudaFuncSetAttribute(chain_long_kernel<kMaxOpsLarge, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, chain_long_smem_bytes<0>()));
        ELG_CK(cudaFuncSetAttribute(chain_long_kernel<kMaxOpsLarge, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, chain_long_smem_bytes<1>()));
        ELG_CK(cudaFuncSetAttribute(chain_long_kernel<kMaxOpsLarge, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, chain_long_smem_bytes<2>()));
        ELG_CK(cudaFuncSetAttribute(chain_long_kernel<kMaxOpsLarge, 3>, cudaFuncAttributeMaxDynamicSharedMemorySize, chain_long_smem_bytes<3>()));
        ELG_CK(cudaFuncSetAttribute(chain_ring_kernel<kMaxOpsSmall>, cudaFuncAttributeMaxDynamicSharedMemorySize, chain_ring_smem_bytes()));
        ELG_CK(cudaFuncSetAttribute(compact_kernel<kMaxOpsSmall, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, compact_smem_bytes()));
        ELG_CK(cudaFuncSetAttribute(compact_kernel<kMaxOpsSmall, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, compact_smem_bytes()));
        ELG_CK(cudaFuncSetAttribute(compact_kernel<kMaxOpsSmall, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, compact_smem_bytes()));
        done = true;
    }
    return ELG_OK;
}

int32_t hist_setup_once() {
    static bool done = false;
    if (!done) {
        ELG_CK(cudaFuncSetAttribute(hist_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, kHistSmemBins * 4));
        ELG_CK(cudaFuncSetAttribute(hist_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kHistSmemBins * 4));
        ELG_CK(cudaFuncSetAttribute(dipole_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, kDipoleSmemBins * 36));
        done = true;
    }
    return ELG_OK;
}

}  // namespace

// =====================================================================================================
extern "C" const char* elg_version(void) { return "elg 0.2 (sm_100a)"; }
extern "C" const char* elg_last_error(void) { return g_err.c_str(); }
extern "C" int64_t elg_launch_count(void) { return g_launches.load(); }
extern "C" int64_t elg_soa_stride(int64_t n0) { return n0 <= 0 ? 32 : align_up(n0, 32); }
extern "C" int64_t elg_soa_bytes(int64_t n0) { return 7 * elg_soa_stride(n0) * 8; }

// ------------------------------------------------------------------------------------- beamline
extern "C" int32_t elg_beamline_load(elg_beamline** out, const elg_element* elems, int64_t n_elems, int32_t ring) {
    if (!out || n_elems < 0 || (n_elems > 0 && !elems)) return fail(ELG_EINVAL, "elg_beamline_load: bad arguments");
    elg_beamline* bl = new (std::nothrow) elg_beamline;
    if (!bl) return fail(ELG_ENOMEM, "elg_beamline_load: out of host memory");
    bl->ring = ring;
    bl->e.assign(elems, elems + n_elems);
    bl->R.resize(n_elems); bl->C.resize(n_elems); bl->table.resize(n_elems); bl->T.resize(n_elems); bl->U.resize(n_elems);
    bl->res.resize(n_elems); bl->table_off.assign(n_elems, 0);
    bl->s_design.resize(n_elems + 1);
    bl->serial = ++g_bl_serial;
    double s = 0.0;                                         // G8: sequential ascending fp64 sum
    for (int64_t k = 0; k < n_elems; k++) {
        elg_element& e = bl->e[k];
        bl->s_design[k] = s;
        const char* why = nullptr;
        switch (e.type) {
            case ELG_DRIFT:
                if (!std::isfinite(e.L)) why = "DRIFT: L not finite"; else s = s + e.L;
                break;
            case ELG_MATRIX: case ELG_MATRIX2: case ELG_MATRIX3:
                if (!e.R) { why = "MATRIX: R is NULL"; break; }
                if (e.type != ELG_MATRIX && !e.T) { why = "MATRIX2/3: T is NULL"; break; }
                if (e.type == ELG_MATRIX3 && !e.U) { why = "MATRIX3: U is NULL"; break; }
                bl->R[k].assign(e.R, e.R + 36); e.R = bl->R[k].data();
                if (e.C) { bl->C[k].assign(e.C, e.C + 6); e.C = bl->C[k].data(); s = s + e.C[4]; }
                if (e.type != ELG_MATRIX) { bl->T[k].assign(e.T, e.T + 126); e.T = bl->T[k].data(); }
                if (e.type == ELG_MATRIX3) { bl->U[k].assign(e.U, e.U + 336); e.U = bl->U[k].data(); }
                break;
            case ELG_RFKICK:
                if (!std::isfinite(e.V) || !std::isfinite(e.f) || !std::isfinite(e.phi)) why = "RFKICK: V, f, phi must be finite";
                break;
            case ELG_RCOL: case ELG_ECOL:
                if (!(e.ax > 0.0) || !(e.ay > 0.0)) why = "aperture: ax, ay must be > 0";
                break;
            case ELG_WAKE: case ELG_HISTO: case ELG_TRWAKE:
                if (e.nb < 2) { why = "WAKE/HISTO: nb < 2"; break; }
                if (e.nb > (1 << 24)) { why = "WAKE/HISTO: nb > 2^24"; break; }
                if (e.window < ELG_WIN_EXPLICIT || e.window > ELG_WIN_AUTO_TABLE) { why = "WAKE/HISTO: bad window mode"; break; }
                if (e.window == ELG_WIN_EXPLICIT && (!(e.dt > 0.0) || !std::isfinite(e.t_lo_rel))) { why = "EXPLICIT window: dt > 0 and finite t_lo_rel required"; break; }
                if (e.nb > bl->nb_max) bl->nb_max = e.nb;
                if (e.type == ELG_TRWAKE && e.wake == ELG_WAKE_RESONATOR) { why = "TRWAKE: wake kind must be RESONATOR_T or TABLE"; break; }
                if (e.type == ELG_WAKE && e.wake == ELG_WAKE_RESONATOR_T) { why = "WAKE: RESONATOR_T is a transverse wake"; break; }
                if (e.type == ELG_TRWAKE && e.wake == ELG_WAKE_RESONATOR_T) {
                    if (!(e.Q > 0.5) || !(e.f > 0.0) || !std::isfinite(e.Rs)) { why = "resonator: Q > 1/2, f > 0, finite Rs required"; break; }
                    const double wr = kTwoPi * e.f;                      // G34, same expressions as the definition
                    ResConst rc;
                    rc.alpha = wr / (2.0 * e.Q);
                    rc.wbar = std::sqrt(wr * wr - rc.alpha * rc.alpha);
                    rc.kloss = (wr * e.Rs / e.Q) * (wr / rc.wbar);       // amplitude
                    rc.ratio = 0.0;
                    bl->res[k] = rc;
                } else if (e.type == ELG_WAKE || e.type == ELG_TRWAKE) {
                    if (e.type == ELG_TRWAKE && e.wake == ELG_WAKE_RESONATOR_REC) { why = "TRWAKE: wake kind must be RESONATOR_T or TABLE"; break; }
                    if (e.wake == ELG_WAKE_RESONATOR || e.wake == ELG_WAKE_RESONATOR_REC) {
                        if (!(e.Q > 0.5) || !(e.f > 0.0) || !std::isfinite(e.Rs)) { why = "resonator: Q > 1/2, f > 0, finite Rs required"; break; }
                        // G12, same expressions as the definition, evaluated once here
                        const double wr = kTwoPi * e.f;
                        ResConst rc;
                        rc.kloss = wr * e.Rs / (2.0 * e.Q);
                        rc.alpha = wr / (2.0 * e.Q);
                        rc.wbar = std::sqrt(wr * wr - rc.alpha * rc.alpha);
                        rc.ratio = rc.alpha / rc.wbar;
                        bl->res[k] = rc;
                    } else if (e.wake == ELG_WAKE_TABLE) {
                        if (!e.table || e.n_table < 1 || !(e.dt_table > 0.0)) { why = "table wake: table, n_table >= 1, dt_table > 0 required"; break; }
                        bl->table[k].assign(e.table, e.table + e.n_table); e.table = bl->table[k].data();
                        bl->table_off[k] = bl->table_total;
                        bl->table_total += e.n_table;
                    } else { why = "WAKE: bad wake kind"; break; }
                }
                if (!why && e.type != ELG_HISTO && e.window == ELG_WIN_AUTO_TABLE && e.wake != ELG_WAKE_TABLE) why = "AUTO_TABLE window needs a table wake";
                break;
            default: why = "unknown element type";
        }
        if (why) {
            char buf[160];
            std::snprintf(buf, sizeof buf, "elg_beamline_load: element %lld: %s", (long long)k, why);
            delete bl;
            return fail(ELG_EINVAL, buf);
        }
    }
    bl->s_design[n_elems] = s;
    bl->length = s;
    *out = bl;
    return ELG_OK;
}
extern "C" void elg_beamline_destroy(elg_beamline* bl) { delete bl; }
extern "C" int64_t elg_beamline_n_elements(const elg_beamline* bl) { return bl ? (int64_t)bl->e.size() : 0; }
extern "C" double elg_beamline_length(const elg_beamline* bl) { return bl ? bl->length : 0.0; }
extern "C" double elg_beamline_s_design(const elg_beamline* bl, int64_t k) {
    if (!bl || k < 0 || k > (int64_t)bl->e.size()) return NAN;
    return bl->s_design[k];
}

// ------------------------------------------------------------------------------------- bunch
extern "C" int32_t elg_workspace_bytes(int64_t n0, const elg_beamline* bl, int64_t lost_capacity, int64_t* bytes) {
    if (n0 < 0 || lost_capacity < 0 || !bytes) return fail(ELG_EINVAL, "elg_workspace_bytes: bad arguments");
    long long nb_cap, table_cap;
    caps_for(bl, &nb_cap, &table_cap);
    *bytes = layout(n0, nb_cap, table_cap, lost_capacity).total;
    return ELG_OK;
}

extern "C" int32_t elg_bunch_rewind(elg_bunch* b) {
    if (!b) return fail(ELG_EINVAL, "elg_bunch_rewind: NULL bunch");
    launch_k(init_state_kernel, 1, 1, 0, b->stream, b->st, b->n0);
    g_launches++;
    ELG_CK(cudaGetLastError());
    b->cur_buf = 0; b->cur_slot = 0; b->turn = 0; b->rec_count = 0;
    return ELG_OK;
}

extern "C" int32_t elg_bunch_create(elg_bunch** out, int64_t n0, void* d_soa, void* d_work, int64_t work_bytes,
                                    const elg_beamline* sized_for, int64_t lost_capacity, double p0c, double mc2, double charge, void* stream) {
    if (!out || n0 < 0 || n0 >= (1LL << 31) || !d_soa || !d_work || lost_capacity < 0 || !(p0c > 0.0) || !(mc2 > 0.0))
        return fail(ELG_EINVAL, "elg_bunch_create: bad arguments (0 <= n0 < 2^31, non-NULL buffers, p0c, mc2 > 0)");
    if (((uintptr_t)d_soa & 255) || ((uintptr_t)d_work & 255))
        return fail(ELG_EINVAL, "elg_bunch_create: d_soa and d_work must be 256-byte aligned");
    long long nb_cap, table_cap;
    caps_for(sized_for, &nb_cap, &table_cap);
    const WorkLayout L = layout(n0, nb_cap, table_cap, lost_capacity);
    if (work_bytes < L.total) return fail(ELG_ECAPACITY, "elg_bunch_create: workspace smaller than elg_workspace_bytes");
    int sms = 0;
    { int32_t rc = device_sms(&sms); if (rc != ELG_OK) return rc; }
    elg_bunch* b = new (std::nothrow) elg_bunch;
    if (!b) return fail(ELG_ENOMEM, "elg_bunch_create: out of host memory");
    b->n0 = n0; b->stride = elg_soa_stride(n0); b->lost_cap = lost_capacity; b->work_bytes = work_bytes;
    b->d_soa = (char*)d_soa; b->d_work = (char*)d_work; b->stream = (cudaStream_t)stream;
    b->p0c = p0c; b->mc2 = mc2; b->charge = charge;
    {   // G7, G9, G30: unfused, in this order
        const double e2 = p0c * p0c + mc2 * mc2;
        b->beta0 = p0c / std::sqrt(e2);
        b->inv_bc = 1.0 / (b->beta0 * kCLight);
        b->inv_E = 1.0 / (b->beta0 * p0c);
        b->q_macro = (n0 > 0) ? charge / (double)n0 : 0.0;     // G15
    }
    b->nb_cap = nb_cap; b->table_cap = table_cap;
    char* w = b->d_work;
    b->st = (DevState*)(w + L.off_state);
    b->soaB = w + L.off_soaB;
    b->tile_status = (unsigned long long*)(w + L.off_status);
    b->mm_partial = (double*)(w + L.off_mm);
    b->mom_partial = (double*)(w + L.off_mom);
    b->records = (double*)(w + L.off_rec);
    b->counts = (unsigned int*)(w + L.off_counts);
    b->W = (double*)(w + L.off_W);
    b->V = (double*)(w + L.off_V);
    b->dacc = (unsigned long long*)(w + L.off_dacc);
    b->D = (double*)(w + L.off_D);
    b->Vt = (double*)(w + L.off_Vt);
    b->table = (double*)(w + L.off_table);
    b->lost_id = (long long*)(w + L.off_lost_id);
    b->lost_te = (long long*)(w + L.off_lost_te);
    b->lost_v = (double*)(w + L.off_lost_v);
    b->sms = sms;
    int32_t rc = ELG_OK;
    if (rc == ELG_OK) rc = long_setup_once();
    if (rc == ELG_OK) rc = hist_setup_once();
    if (rc == ELG_OK) rc = grid_for(moments_kernel, sms, 0, kBlock, &b->grid_mom);
    if (rc != ELG_OK) { delete b; return rc; }
    const char* agg = std::getenv("ELG_HIST_AGGREGATE");
    b->hist_aggregate = agg ? std::atoi(agg) : -1;                 // -1: automatic
    const char* fp = std::getenv("ELG_CHAIN_P");
    b->force_p = fp ? std::atoi(fp) : 0;
    cudaError_t ce = cudaMemsetAsync(b->st, 0, sizeof(DevState), b->stream);       // incl. the work counters of elg_profile_read
    if (ce == cudaSuccess) ce = cudaMemsetAsync(b->tile_status, 0, (b->stride / kStatusTile + 2) * 8, b->stream);
    if (ce != cudaSuccess) { delete b; return fail(ELG_ECUDA, std::string("cudaMemsetAsync: ") + cudaGetErrorString(ce)); }
    rc = elg_bunch_rewind(b);
    if (rc != ELG_OK) { delete b; return rc; }
    *out = b;
    return ELG_OK;
}
extern "C" void elg_bunch_destroy(elg_bunch* b) {
    if (b) {
        cudaStreamSynchronize(b->stream);
        b->prof_drain();
        for (cudaEvent_t e : b->prof_pool) cudaEventDestroy(e);
        for (cudaEvent_t e : b->chunk_ev) cudaEventDestroy(e);
        if (b->entry_ev) cudaEventDestroy(b->entry_ev);
        if (b->copy_stream) cudaStreamDestroy(b->copy_stream);
    }
    delete b;
}

extern "C" int32_t elg_profile_enable(elg_bunch* b, int32_t on) {
    if (!b) return fail(ELG_EINVAL, "elg_profile_enable: NULL bunch");
    b->prof_on = on != 0;
    return ELG_OK;
}

extern "C" int32_t elg_profile_read(elg_bunch* b, int64_t* h_launches, double* h_ms, double* h_bytes, double* h_flops) {
    if (!b || !h_launches || !h_ms) return fail(ELG_EINVAL, "elg_profile_read: bad arguments");
    unsigned long long work[16];
    ELG_CK(cudaMemcpyAsync(work, b->st->work, sizeof work, cudaMemcpyDeviceToHost, b->stream));
    ELG_CK(cudaMemsetAsync(b->st->work, 0, sizeof work, b->stream));
    ELG_CK(cudaStreamSynchronize(b->stream));
    b->prof_drain();
    for (int k = 0; k < ELG_K_COUNT; k++) {
        h_launches[k] = b->prof_launches[k]; h_ms[k] = b->prof_ms[k];
        if (h_bytes) h_bytes[k] = (double)work[2 * k];
        if (h_flops) h_flops[k] = (double)work[2 * k + 1];
        b->prof_launches[k] = 0; b->prof_ms[k] = 0.0;
    }
    return ELG_OK;
}

// The fp64 roofline denominator, measured: a DFMA-only kernel (8 independent chains per thread, register operands) on
// two blocks of 256 threads per SM, timed with CUDA events on `stream`.  d_scratch: >= 2048 bytes of device memory.
extern "C" int32_t elg_dbg_fp64_peak(double* d_scratch, int64_t iters, double* h_tflops, double* h_ms, void* stream) {
    if (!d_scratch || iters < 1 || !h_tflops) return fail(ELG_EINVAL, "elg_dbg_fp64_peak: bad arguments");
    int sms = 0;
    { int32_t rc = device_sms(&sms); if (rc != ELG_OK) return rc; }
    cudaStream_t st = (cudaStream_t)stream;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    ELG_CK(cudaEventCreate(&e0));
    ELG_CK(cudaEventCreate(&e1));
    const int grid = 2 * sms;
    float ms = 0.f;
    for (int rep = 0; rep < 4; rep++) {                                // rep 0 warms the clocks up; best of the other three
        ELG_CK(cudaEventRecord(e0, st));
        launch_k(fp64_peak_kernel, grid, kBlock, 0, st, d_scratch, iters, 0.999, 1e-7);
        ELG_CK(cudaEventRecord(e1, st));
        g_launches++;
        ELG_CK(cudaGetLastError());
        ELG_CK(cudaEventSynchronize(e1));
        float t = 0.f;
        ELG_CK(cudaEventElapsedTime(&t, e0, e1));
        if (rep >= 1 && (ms == 0.f || t < ms)) ms = t;
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    const double fma = (double)grid * kBlock * kPeakIlp * kPeakUnroll * (double)iters;
    *h_tflops = 2.0 * fma / ((double)ms * 1e-3) / 1e12;
    if (h_ms) *h_ms = (double)ms;
    return ELG_OK;
}

extern "C" int32_t elg_bunch_upload(elg_bunch* b, const double* const h_coords[6], const int64_t* h_ids) {
    if (!b || !h_coords) return fail(ELG_EINVAL, "elg_bunch_upload: bad arguments");
    for (int c = 0; c < 6; c++) {
        if (!h_coords[c]) return fail(ELG_EINVAL, "elg_bunch_upload: NULL coordinate array");
        ELG_CK(cudaMemcpyAsync(b->coord(0, c), h_coords[c], b->n0 * 8, cudaMemcpyHostToDevice, b->stream));
    }
    if (h_ids) ELG_CK(cudaMemcpyAsync(b->ids(0), h_ids, b->n0 * 8, cudaMemcpyHostToDevice, b->stream));
    else if (b->n0 > 0) {
        launch_k(iota_kernel, b->sms * 4, kBlock, 0, b->stream, b->ids(0), b->n0);
        g_launches++;
        ELG_CK(cudaGetLastError());
    }
    return elg_bunch_rewind(b);
}

// =====================================================================================================
// Tracking: the beamline is cut into fused runs (north_star part 1).  Maps accumulate in a pending list
// and are launched as ONE chain kernel when something needs the particles in memory: an aperture (which
// becomes the run's terminator and compacts), a WAKE/HISTO (needs min/max of s: fused epilogue), a
// moments record, more ops than one parameter block holds, or the end of the call.  The wake kick is
// not a pass of its own: it is queued as the first op of the next run.
// With b == nullptr the planner only counts launches (elg_beamline_launches_per_turn; CPU-testable).
// =====================================================================================================
namespace {

struct Tracker {
    elg_bunch* b;
    const elg_beamline* bl;
    elg_track_opts* o;
    std::vector<HostOp> pending;
    int kick_nb = 0, kick_interp = 0;
    int tk_nb = 0, tk_interp = 0;
    long long range_lo = 0, range_hi = -1;   // particle range of the chain launches (pipelined upload), -1: all live
    int mm_slot = 0;                         // min/max partials of chunk c go to slot c of the partial array
    bool mm_valid = false;
    long long launches = 0;
    int32_t rc = ELG_OK;
    long long rec_total = 0;       // records taken in this call
    long long rec_flushed = 0;     // of which already copied to the host
    int mm_grid = 0;               // blocks of the launch that produced the current min/max partials

    bool ok() const { return rc == ELG_OK; }
    void count() { launches++; if (b) g_launches++; }
    void check(cudaError_t e, const char* what) {
        if (e != cudaSuccess && rc == ELG_OK) rc = fail(ELG_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
    }

    int hist_grid(int smem_bins) {                                    // resident blocks of hist_kernel for this much shared memory
        auto it = b->hist_grids.find(smem_bins);
        if (it != b->hist_grids.end()) return it->second;
        int occ = 0;
        check(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, hist_kernel<false>, kBlock, (size_t)smem_bins * 4), "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
        if (occ < 1) occ = 1;
        const int g = occ * b->sms;
        b->hist_grids[smem_bins] = g;
        return g;
    }

    int dipole_grid(int smem_bins) {
        auto it = b->dipole_grids.find(smem_bins);
        if (it != b->dipole_grids.end()) return it->second;
        int occ = 0;
        check(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dipole_hist_kernel, kBlock, (size_t)smem_bins * 36), "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
        if (occ < 1) occ = 1;
        const int g = occ * b->sms;
        b->dipole_grids[smem_bins] = g;
        return g;
    }

    // blocks of a persistent grid = resident blocks per SM x SMs, looked up once per kernel
    int cached_grid(const void* kernel, int smem, int threads = kBlock) {
        auto it = b->grids.find(kernel);
        if (it != b->grids.end()) return it->second;
        int occ = 0;
        check(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kernel, threads, smem), "cudaOccupancyMaxActiveBlocksPerMultiprocessor");
        if (occ < 1 && rc == ELG_OK) rc = fail(ELG_ECUDA, "kernel does not fit on an SM");
        long long g = (long long)occ * b->sms;
        if (g > kMaxGrid) g = kMaxGrid / b->sms * b->sms;
        b->grids[kernel] = (int)g;
        return (int)g;
    }

    // chain_ring_kernel takes the short runs that are nothing but DRIFT / MATRIX maps (the purely HBM-bound ones: 1.626 ->
    // 1.584 ms at 1e8 particles); with a wake or RF kick in the run the register-held form measured as fast or faster
    // (cfg2's KICK + DRIFT at 1e7 particles: 0.163 vs 0.174 ms per pass)
    bool use_ring() const {
        if (!ring_enabled()) return false;
        for (const HostOp& op : pending)
            if (op.type != OP_DRIFT && op.type != OP_MATRIX) return false;
        return !pending.empty();
    }

    // EXT: 0 basic maps, 1 + MATRIX2 / TKICK, 2 + MATRIX3, 3 pattern matrices.  MOM: moment epilogue (record slot rec_count)
    template <int MAXOPS, bool COMPACT, int P, int EXT, bool MOM = false>
    void launch_chain(int ap_type, double ap_x, double ap_y, long long te_code, bool want_mm, unsigned rmask, unsigned wmask) {
        count();
        if (!b) return;
        ChainArgs<MAXOPS> a;
        ChainCommon& c = a.c;
        const int src = b->cur_buf, dst = COMPACT ? (b->cur_buf ^ 1) : b->cur_buf;
        for (int k = 0; k < 6; k++) { c.src[k] = b->coord(src, k); c.dst[k] = b->coord(dst, k); }
        c.id_src = b->ids(src); c.id_dst = b->ids(dst);
        c.st = b->st; c.cur = b->cur_slot; c.n_ops = (int)pending.size();
        c.rmask = rmask; c.wmask = wmask;
        c.ap_type = ap_type; c.ap_x = ap_x; c.ap_y = ap_y;
        c.lost_id = b->lost_id; c.lost_te = b->lost_te; c.lost_v = b->lost_v; c.lost_cap = b->lost_cap; c.te_code = te_code;
        c.tile_status = b->tile_status;
        if (COMPACT) b->epoch = (b->epoch + 1) & 0x3fffffffu;
        if (COMPACT && b->epoch == 0) {                               // epoch wrapped: stale tags could alias
            check(cudaMemsetAsync(b->tile_status, 0, (b->stride / kStatusTile + 2) * 8, b->stream), "cudaMemsetAsync");
            b->epoch = 1;
        }
        c.epoch = b->epoch;
        c.want_minmax = want_mm ? 1 : 0;
        c.range_lo = range_lo; c.range_hi = range_hi;
        c.V = b->V; c.nb = kick_nb; c.interp = kick_interp;
        c.Vx = b->Vt; c.Vy = b->Vt + tk_nb; c.t_nb = tk_nb; c.t_interp = tk_interp;
        c.mom_partial = b->mom_partial; c.mom_record = b->records + 43 * b->rec_count;
        c.prof_kind = b->prof_on ? (MAXOPS == kMaxOpsLarge ? ELG_K_CHAIN_LONG : (COMPACT ? ELG_K_CHAIN_COMPACT : ELG_K_CHAIN)) : -1;
        // a compacting run moves all seven arrays (56 B in, 56 B out); the others only the coordinates they read / write
        c.bytes_pp = COMPACT ? 112u : 8u * (unsigned)(__builtin_popcount(rmask) + __builtin_popcount(wmask));
        c.flops_pp = MOM ? 60u : 0u;                                  // algorithmic flops per particle
        for (const HostOp& op : pending) {
            switch (op.type) {
                case OP_MATRIX: c.flops_pp += 72u; break;
                case OP_MATRIX_UNC: c.flops_pp += 40u; break;
                case OP_MATRIX2: c.flops_pp += 72u + 21u + 252u; break;
                case OP_MATRIX3: c.flops_pp += 72u + 21u + 252u + 56u + 672u; break;
                case OP_DRIFT: c.flops_pp += 11u; break;
                case OP_RFKICK: c.flops_pp += 6u; break;
                case OP_KICK: c.flops_pp += 10u; break;
                case OP_TKICK: c.flops_pp += 14u; break;
                case OP_KICK3: c.flops_pp += 18u; break;
                default: break;
            }
        }
        for (size_t k = 0; k < pending.size(); k++) {
            a.type[k] = pending[k].type;
            std::memcpy(a.coef[k], pending[k].coef, sizeof(double) * 42);
        }
        for (int k = (int)pending.size() - 1; k >= 0; k--)            // lengths of the runs of consecutive MATRIX slots
        {
            const uint8_t ty = pending[k].type;                       // (MATRIX and MATRIX_UNC runs are counted separately)
            const bool run_type = ty == OP_MATRIX || ty == OP_MATRIX_UNC;
            const bool same_next = (size_t)k + 1 < pending.size() && pending[k + 1].type == ty;
            a.mat_run[k] = !run_type ? 0 : (uint8_t)(1 + (same_next ? a.mat_run[k + 1] : 0));
        }
        int grid = 0;
        if constexpr (MAXOPS == kMaxOpsLarge) grid = cached_grid((const void*)chain_long_kernel<MAXOPS, EXT>, chain_long_smem_bytes<EXT>(), LongCfg<EXT>::NT);
        else if constexpr (COMPACT) {
            grid = cached_grid((const void*)compact_kernel<MAXOPS, (EXT != 0), MOM>, compact_smem_bytes(), kC2Threads);
            if (grid > kCompactMaxGrid) grid = kCompactMaxGrid;      // kPoll status words per thread
        } else if constexpr (P == 2 && EXT == 0 && !MOM) {
            if (use_ring()) grid = cached_grid((const void*)chain_ring_kernel<MAXOPS>, chain_ring_smem_bytes(), kCrThreads);
            else grid = cached_grid((const void*)chain_kernel<MAXOPS, P, false, MOM>, 0);
        } else grid = cached_grid((const void*)chain_kernel<MAXOPS, P, (EXT != 0), MOM>, 0);
        if (!ok()) return;
        if ((long long)(mm_slot + 1) * grid > kMmPartials) { rc = fail(ELG_ECAPACITY, "elg_upload_and_track: too many chunks for the min/max partial slots"); return; }
        c.mm_partial = b->mm_partial + 2LL * mm_slot * grid;          // one slot of partials per chunk
        if (want_mm) mm_grid = (mm_slot + 1) * grid;
        {
            ProfScope ps(b, MAXOPS == kMaxOpsLarge ? ELG_K_CHAIN_LONG : (COMPACT ? ELG_K_CHAIN_COMPACT : ELG_K_CHAIN));
            if constexpr (MAXOPS == kMaxOpsLarge)
                launch_k(chain_long_kernel<MAXOPS, EXT>, grid, LongCfg<EXT>::NT, chain_long_smem_bytes<EXT>(), b->stream, a);
            else if constexpr (COMPACT)
            {
                cudaLaunchConfig_t cfg{};                        // cooperative: every block resident (static tiles)
                cfg.gridDim = dim3(grid); cfg.blockDim = dim3(kC2Threads); cfg.dynamicSmemBytes = compact_smem_bytes(); cfg.stream = b->stream;
                cudaLaunchAttribute attr[2];
                attr[0].id = cudaLaunchAttributeCooperative; attr[0].val.cooperative = 1;
                attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization; attr[1].val.programmaticStreamSerializationAllowed = 1;
                cfg.attrs = attr; cfg.numAttrs = pdl_enabled() ? 2 : 1;
                check(cudaLaunchKernelEx(&cfg, compact_kernel<MAXOPS, (EXT != 0), MOM>, a), "compact_kernel cooperative launch");
            }
            else if constexpr (P == 2 && EXT == 0 && !MOM) {
                if (use_ring()) launch_k(chain_ring_kernel<MAXOPS>, grid, kCrThreads, chain_ring_smem_bytes(), b->stream, a);
                else launch_k(chain_kernel<MAXOPS, P, false, MOM>, grid, kBlock, 0, b->stream, a);
            }
            else
                launch_k(chain_kernel<MAXOPS, P, (EXT != 0), MOM>, grid, kBlock, 0, b->stream, a);
        }
        check(cudaGetLastError(), "chain_kernel launch");
        if (COMPACT) { b->cur_buf ^= 1; b->cur_slot ^= 1; }
    }

    // launch the pending maps (+ aperture terminator, + min/max epilogue, + moment epilogue when a record follows)
    bool want_mom = false;         // set by moments_record(): the run being flushed is followed by a record
    bool mom_fused = false;        // ... and this flush has taken it in its epilogue
    void flush(int ap_type, double ap_x, double ap_y, long long te_code, bool want_mm) {
        if (!ok()) return;
        if (ap_type == AP_NONE && pending.empty() && !want_mm) return;
        // a long run that ends in an aperture: the maps go through the fp64-bound long-run kernel, the
        // aperture and the compaction follow as a run of their own (112 B per particle more, rare)
        if (ap_type != AP_NONE && pending.size() > (size_t)kMaxOpsSmall) {
            const bool keep = want_mom;
            want_mom = false;
            flush(AP_NONE, 0, 0, 0, false);
            want_mom = keep;
        }
        unsigned rmask = 0, wmask = 0;
        for (const HostOp& op : pending) {
            switch (op.type) {
                case OP_DRIFT: rmask |= 0x1F; wmask |= 0x15; break;           // reads x x' y y' s, writes x y s
                case OP_MATRIX: case OP_MATRIX2: case OP_MATRIX3: case OP_MATRIX_UNC: rmask |= 0x3F; wmask |= 0x3F; break;
                case OP_RFKICK: case OP_KICK: rmask |= 0x30; wmask |= 0x20; break;   // reads s delta, writes delta
                case OP_TKICK: rmask |= 0x1A; wmask |= 0x0A; break;                  // reads x' y' s, writes x' y'
                case OP_KICK3: rmask |= 0x3A; wmask |= 0x2A; break;                  // both
            }
        }
        if (want_mm) rmask |= 0x10;
        // the long-run kernel (coefficients as uniform operands, 6 particles per thread) also takes the short runs that
        // are already fp64-bound: from 5 matrices on it beats the parameter-bank kernel (bench.py p3 sweep)
        int n_mat_run = 0;
        for (const HostOp& op : pending) n_mat_run += (op.type == OP_MATRIX || op.type == OP_MATRIX_UNC) + 4 * (op.type == OP_MATRIX2);
        const bool large = pending.size() > (size_t)kMaxOpsSmall || (ap_type == AP_NONE && n_mat_run >= kMatricesForLong);
        const bool compact = ap_type != AP_NONE;
        // particles per thread: 2 while the run is HBM-bound; 4 once it holds enough MATRIX maps for the
        // coefficient fetches (one per 2 particles) to matter
        int n_mat = 0;
        for (const HostOp& op : pending) n_mat += (op.type == OP_MATRIX || op.type == OP_MATRIX_UNC) + 4 * (op.type == OP_MATRIX2) + 12 * (op.type == OP_MATRIX3);
        bool p4 = n_mat >= kMatricesForP4;
        if (b && b->force_p == 2) p4 = false;
        if (b && b->force_p == 4) p4 = true;
        int ext = 0;                                                  // rarely used maps: higher EXT instantiations
        bool has_unc = false;
        for (const HostOp& op : pending) {
            if (op.type == OP_MATRIX2 || ((op.type == OP_TKICK || op.type == OP_KICK3) && (large || compact || !ELG_TKICK_BASE))) ext = ext < 1 ? 1 : ext;
            if (op.type == OP_MATRIX3) ext = 2;
            has_unc = has_unc || op.type == OP_MATRIX_UNC;
        }
        if (has_unc) {
            if (large && ext == 0) ext = 3;                           // the pattern level of the long-run kernel
            else                                                      // short or mixed run: apply them densely
                for (HostOp& op : pending)
                    if (op.type == OP_MATRIX_UNC) { op.type = OP_MATRIX; std::memcpy(op.coef, op.dense, sizeof op.coef); }
        }
        // moment epilogue: short runs of the basic maps over the whole live set (the record needs all six coordinates)
        const bool mom = want_mom && !large && ext == 0 && range_hi < 0;
        if (mom) { rmask = 0x3F; mom_fused = true; }
#define ELG_LAUNCH(M, C, PP, E) launch_chain<M, C, PP, E>(ap_type, ap_x, ap_y, te_code, want_mm, rmask, wmask)
#define ELG_LAUNCH_MOM(M, C, PP) launch_chain<M, C, PP, 0, true>(ap_type, ap_x, ap_y, te_code, want_mm, rmask, wmask)
        if (mom) {
            if (compact) ELG_LAUNCH_MOM(kMaxOpsSmall, true, 2);
            else ELG_LAUNCH_MOM(kMaxOpsSmall, false, 2);              // (27 sums + 4 particles per thread would spill)
        }
        else if (large) {
            if (ext == 3) ELG_LAUNCH(kMaxOpsLarge, false, 0, 3);
            else if (ext == 2) ELG_LAUNCH(kMaxOpsLarge, false, 0, 2);
            else if (ext == 1) ELG_LAUNCH(kMaxOpsLarge, false, 0, 1);
            else ELG_LAUNCH(kMaxOpsLarge, false, 0, 0);
        }
        else if (compact) { if (ext) ELG_LAUNCH(kMaxOpsSmall, true, 2, 1); else ELG_LAUNCH(kMaxOpsSmall, true, 2, 0); }
        else if (p4) { if (ext) ELG_LAUNCH(kMaxOpsSmall, false, 4, 1); else ELG_LAUNCH(kMaxOpsSmall, false, 4, 0); }
        else         { if (ext) ELG_LAUNCH(kMaxOpsSmall, false, 2, 1); else ELG_LAUNCH(kMaxOpsSmall, false, 2, 0); }
#undef ELG_LAUNCH
#undef ELG_LAUNCH_MOM
        if (compact || (wmask & 0x10)) mm_valid = want_mm;
        else mm_valid = mm_valid || want_mm;
        pending.clear();
    }

    void push(const HostOp& op, int slots = 1) {           // slots: parameter-block slots the op and its continuation take
        if (pending.size() + slots > (size_t)kMaxOpsLarge) flush(AP_NONE, 0, 0, 0, false);
        pending.push_back(op);
    }

    // MATRIX: dense, or (ELG_TRACK_SPARSE_MATRICES) packed for the uncoupled zero pattern when every entry outside it is
    // exactly zero (layout only: the 20 kept coefficients and C in the order matrix_unc_map_uniform reads them)
    void push_matrix(const elg_element& e) {
        HostOp op{};
        op.type = OP_MATRIX;
        std::memcpy(op.coef, e.R, 36 * sizeof(double));
        if (e.C) std::memcpy(op.coef + 36, e.C, 6 * sizeof(double));
        if (o && (o->flags & ELG_TRACK_SPARSE_MATRICES)) {
            static const unsigned char keep[6][6] = {{1, 1, 0, 0, 0, 1}, {1, 1, 0, 0, 0, 1}, {0, 0, 1, 1, 0, 1},
                                                     {0, 0, 1, 1, 0, 1}, {1, 1, 1, 1, 1, 1}, {0, 0, 0, 0, 1, 1}};
            bool fits = true;
            for (int r = 0; r < 6; r++)
                for (int c = 0; c < 6; c++) fits = fits && (keep[r][c] || e.R[6 * r + c] == 0.0);
            if (fits) {
                std::memcpy(op.dense, op.coef, sizeof op.dense);
                const double* R = op.dense; const double* C = op.dense + 36;
                const double packed[28] = {R[0], R[1], R[5], C[0], R[6], R[7], R[11], C[1], R[14], R[15], R[17], C[2],
                                           R[20], R[21], R[23], C[3], R[24], R[25], R[26], R[27], R[28], R[29], C[4], R[34],
                                           R[35], C[5], 0.0, 0.0};
                std::memset(op.coef, 0, sizeof op.coef);
                std::memcpy(op.coef, packed, sizeof packed);
                op.type = OP_MATRIX_UNC;
            }
        }
        push(op);
    }

    void push_higher_order(const elg_element& e) {                    // 4 slots: R, C | Tt[21][6]; MATRIX3: + 8 slots Ut[56][6]
        HostOp op{};
        const bool third = e.type == ELG_MATRIX3;
        op.type = third ? OP_MATRIX3 : OP_MATRIX2;
        std::memcpy(op.coef, e.R, 36 * sizeof(double));
        if (e.C) std::memcpy(op.coef + 36, e.C, 6 * sizeof(double));
        push(op, third ? 12 : 4);
        for (int part = 0; part < 3; part++) {
            HostOp t{};
            t.type = OP_CONT;
            for (int j = 0; j < 42; j++) {                           // layout only: pair-major transpose of T
                const int q = (42 * part + j) / 6, r = (42 * part + j) % 6;
                t.coef[j] = e.T[21 * r + q];
            }
            pending.push_back(t);
        }
        for (int part = 0; third && part < 8; part++) {
            HostOp t{};
            t.type = OP_CONT;
            for (int j = 0; j < 42; j++) {                           // layout only: triple-major transpose of U
                const int q = (42 * part + j) / 6, r = (42 * part + j) % 6;
                t.coef[j] = e.U[56 * r + q];
            }
            pending.push_back(t);
        }
    }

    // one record (G26) of the live set as it is after the pending maps (and the aperture ap_type, if any): taken in the
    // epilogue of the run that is flushed when that is possible, else by a pass of moments_kernel
    void moments_record(int ap_type = AP_NONE, double ap_x = 0, double ap_y = 0, long long te_code = 0, bool want_mm = false) {
        if (!ok()) return;
        if (b && b->rec_count == kRecCap) flush_records();
        want_mom = true; mom_fused = false;
        flush(ap_type, ap_x, ap_y, te_code, want_mm);
        want_mom = false;
        if (!ok()) return;
        rec_total++;
        if (mom_fused) { if (b) b->rec_count++; return; }
        count();
        if (!b) return;
        MomArgs m;
        for (int k = 0; k < 6; k++) m.src[k] = b->coord(b->cur_buf, k);
        m.st = b->st; m.cur = b->cur_slot; m.partial = b->mom_partial; m.prof_kind = b->prof_on ? ELG_K_MOMENTS : -1;
        m.record = b->records + 43 * b->rec_count;
        {
            ProfScope ps(b, ELG_K_MOMENTS);
            launch_k(moments_kernel, b->grid_mom, kBlock, 0, b->stream, m);
        }
        check(cudaGetLastError(), "moments_kernel launch");
        b->rec_count++;
    }

    void flush_records() {             // device ring -> host (drops what does not fit)
        if (!b || b->rec_count == 0) return;
        if (o && o->records) {
            long long room = o->capacity_records - rec_flushed;
            long long m = b->rec_count < room ? b->rec_count : room;
            if (m > 0) check(cudaMemcpyAsync(o->records + 43 * rec_flushed, b->records, m * 43 * 8, cudaMemcpyDeviceToHost, b->stream), "records D2H");
            check(cudaStreamSynchronize(b->stream), "cudaStreamSynchronize");
        }
        rec_flushed += b->rec_count;
        b->rec_count = 0;
    }

    // WAKE / HISTO / TRWAKE.  A WAKE directly followed by a TRWAKE with the same binning (the RFCW composite of
    // "RFCW, which is a combination of RFCA, WAKE, TRWAKE ...") shares ONE window and ONE histogram
    // pass (the dipole histogram also yields the counts: 24 B per particle instead of 8 + 24), and both kicks
    // wait in the pending list for the next fused run, so a cavity costs one pass over the particles.
    bool skip_next = false;

    bool mergeable(long long k) const {
        if (k + 1 >= (long long)bl->e.size()) return false;
        const elg_element& w = bl->e[k];
        const elg_element& t = bl->e[k + 1];
        if (w.type != ELG_WAKE || t.type != ELG_TRWAKE) return false;
        if (o && o->moments_every == ELG_MOM_ELEMENT) return false;
        if (w.nb != t.nb || w.window != t.window) return false;
        if (w.window == ELG_WIN_EXPLICIT && (w.dt != t.dt || w.t_lo_rel != t.t_lo_rel)) return false;
        if (w.window == ELG_WIN_AUTO_TABLE && w.dt_table != t.dt_table) return false;
        return true;
    }

    void wake_or_histo(long long k, double s_here) {
        const elg_element& e = bl->e[k];
        const bool merged = mergeable(k);
        prepare_hist(e, b ? s_here * b->inv_bc : 0.0, e.type == ELG_TRWAKE || merged);
        if (!ok() || e.type == ELG_HISTO) return;
        if (e.type == ELG_WAKE) {
            wake_part(k);
            if (merged) {                                             // the TRWAKE's window and counts are the same
                if (b) stage_out_hist(e.nb);
                else if (o) { o->window_written++; o->hist_written += e.nb; }
                trwake_part(k + 1);
                skip_next = true;
                // both kicks look the same bin up: one op (identical arithmetic per coordinate, one bin_of)
                const size_t np = pending.size();
                if (np >= 2 && pending[np - 2].type == OP_KICK && pending[np - 1].type == OP_TKICK && kick_nb == tk_nb && kick_interp == tk_interp) {
                    pending.pop_back();
                    pending.back().type = OP_KICK3;
                }
            }
        } else {
            trwake_part(k);
        }
    }

    // min/max epilogue of the pending run, window, histogram.  t_design: design arrival time at the element (EXPLICIT)
    void prepare_hist(const elg_element& e, double t_design, bool dipole) {
        bool writes_s = false;
        for (const HostOp& op : pending) writes_s = writes_s || op.type == OP_DRIFT || op.type == OP_MATRIX || op.type == OP_MATRIX2 || op.type == OP_MATRIX3 || op.type == OP_MATRIX_UNC;
        const bool need_mm = !mm_valid || writes_s;
        if (!pending.empty() || need_mm) flush(AP_NONE, 0, 0, 0, need_mm);
        if (!ok()) return;
        count();                                                      // window
        count();                                                      // histogram
        if (b) {
            launch_window(e, t_design, dipole);
            if (!ok()) return;
            if (dipole) {                                             // counts + exact dipole sums (G33)
                DipoleArgs d;
                d.s = b->coord(b->cur_buf, 4); d.x = b->coord(b->cur_buf, 0); d.y = b->coord(b->cur_buf, 2);
                d.st = b->st; d.cur = b->cur_slot; d.inv_bc = b->inv_bc; d.nb = e.nb; d.counts = b->counts; d.dacc = b->dacc;
                d.prof_kind = b->prof_on ? ELG_K_HIST : -1;
                // shared memory for the bins this element can occupy: small histograms get more resident blocks
                d.smem_bins = e.nb < kDipoleSmemBins ? (e.nb + 31) / 32 * 32 : kDipoleSmemBins;
                ProfScope ps(b, ELG_K_HIST);
                launch_k(dipole_hist_kernel, dipole_grid(d.smem_bins), kBlock, (size_t)d.smem_bins * 36, b->stream, d);
            } else {
                HistArgs h;
                h.s = b->coord(b->cur_buf, 4); h.st = b->st; h.cur = b->cur_slot; h.n_fixed = -1; h.prof_kind = b->prof_on ? ELG_K_HIST : -1;
                h.inv_bc = b->inv_bc; h.t_lo = 0; h.inv_dt = 0; h.nb = e.nb; h.counts = b->counts;
                h.aggregate = b->hist_aggregate < 0 ? 0 : b->hist_aggregate;
                // one private copy per warp needs 8 nb bins: small histograms take less shared memory and get more
                // resident blocks (more loads in flight)
                h.smem_bins = (8LL * e.nb < kHistSmemBins) ? 8 * e.nb : kHistSmemBins;
                ProfScope ps(b, ELG_K_HIST);
                if (h.aggregate) launch_k(hist_kernel<true>, hist_grid(h.smem_bins), kBlock, h.smem_bins * 4, b->stream, h);
                else launch_k(hist_kernel<false>, hist_grid(h.smem_bins), kBlock, h.smem_bins * 4, b->stream, h);

            }
            check(cudaGetLastError(), "hist_kernel launch");
            stage_out_hist(e.nb);
        } else if (o) { o->window_written++; o->hist_written += e.nb; }
    }

    // window_kernel: min/max partials of the last epilogue -> device-resident window + occupied bin range, zero counts
    void launch_window(const elg_element& e, double t_design, bool dipole) {
        if (e.nb > b->nb_cap) { rc = fail(ELG_ECAPACITY, "elg_track: workspace was sized for fewer bins than this beamline needs"); return; }
        WindowArgs w;
        w.st = b->st; w.cur = b->cur_slot; w.mm_partial = b->mm_partial; w.n_partial = mm_grid;
        w.mode = e.window; w.nb = e.nb; w.t_lo_rel = e.t_lo_rel;
        w.dt_in = (e.window == ELG_WIN_AUTO_TABLE) ? e.dt_table : e.dt;
        w.t_design = t_design; w.inv_bc = b->inv_bc; w.counts = b->counts;
        w.dacc = dipole ? reinterpret_cast<long long*>(b->dacc) : nullptr;
        {
            ProfScope ps(b, ELG_K_WINDOW);
            launch_k(window_kernel, (e.nb + 4 * kBlock - 1) / (4 * kBlock), kBlock, 0, b->stream, w);
        }
        check(cudaGetLastError(), "window_kernel launch");
    }

    void dipole_finalize(int nb) {                                    // fixed-point accumulators -> Dx, Dy (G33)
        ProfScope ps(b, ELG_K_CONV);
        launch_k(dipole_finalize_kernel, (nb + kBlock - 1) / kBlock, kBlock, 0, b->stream, b->dacc, nb, b->D);
        check(cudaGetLastError(), "dipole_finalize_kernel launch");
    }

    // the wake kicks are not passes of their own: they wait in the pending list as the first ops of the next run
    void queue_kick(int nb, int interp) {
        HostOp op{};
        op.type = OP_KICK;
        op.coef[0] = b ? b->inv_bc : 0.0; op.coef[1] = b ? b->inv_E : 0.0;
        pending.push_back(op);
        kick_nb = nb; kick_interp = interp;
    }
    void queue_tkick(int nb, int interp) {
        HostOp op{};
        op.type = OP_TKICK;
        op.coef[0] = b ? b->inv_bc : 0.0; op.coef[1] = b ? b->inv_E : 0.0;
        pending.push_back(op);
        tk_nb = nb; tk_interp = interp;
    }

    void launch_samples(long long k) {
        const elg_element& e = bl->e[k];
        WakeArgs wa;
        wa.st = b->st; wa.dt_fixed = 0.0; wa.kind = e.wake; wa.nb = e.nb;
        const ResConst& r = bl->res[k];
        wa.kloss = r.kloss; wa.alpha = r.alpha; wa.wbar = r.wbar; wa.ratio = r.ratio;
        wa.table = b->table + bl->table_off[k]; wa.n_table = e.n_table; wa.dt_table = e.dt_table; wa.W = b->W;
        {
            ProfScope ps(b, ELG_K_WAKE_SAMPLES);
            launch_k(wake_samples_kernel, (e.nb + kBlock - 1) / kBlock, kBlock, 0, b->stream, wa);
        }
        check(cudaGetLastError(), "wake_samples_kernel launch");
    }

    void wake_part(long long k) {                                     // samples, convolution, queue the kick
        const elg_element& e = bl->e[k];
        count();
        if (e.wake != ELG_WAKE_RESONATOR_REC) count();
        if (b && e.wake == ELG_WAKE_RESONATOR_REC) {                 // O(nb) recurrence: no samples, no convolution (G37)
            const ResConst& r = bl->res[k];
            ConvRecArgs cr;
            cr.counts = b->counts; cr.st = b->st; cr.nb = e.nb; cr.q = b->q_macro;
            cr.kloss = r.kloss; cr.alpha = r.alpha; cr.wbar = r.wbar; cr.ratio = r.ratio; cr.V = b->V;
            {
                ProfScope ps(b, ELG_K_CONV);
                launch_k(conv_rec_kernel, 1, kBlock, 0, b->stream, cr);
            }
            check(cudaGetLastError(), "conv_rec_kernel launch");
            if (o && o->V_out && o->V_written + e.nb <= o->V_capacity)
                check(cudaMemcpyAsync(o->V_out + o->V_written, b->V, (size_t)e.nb * 8, cudaMemcpyDeviceToHost, b->stream), "V D2H");
        } else if (b) {
            launch_samples(k);
            ConvArgs<unsigned int> cv;
            cv.counts = b->counts; cv.W = b->W; cv.st = b->st; cv.nb = e.nb; cv.q = b->q_macro; cv.V = b->V;
            {
                ProfScope ps(b, ELG_K_CONV);
                launch_k(conv_kernel<unsigned int>, (e.nb + kWarps - 1) / kWarps, kBlock, 0, b->stream, cv);
            }
            check(cudaGetLastError(), "conv_kernel launch");
            if (o && o->V_out && o->V_written + e.nb <= o->V_capacity)
                check(cudaMemcpyAsync(o->V_out + o->V_written, b->V, (size_t)e.nb * 8, cudaMemcpyDeviceToHost, b->stream), "V D2H");
        }
        if (o) o->V_written += e.nb;
        queue_kick(e.nb, e.interp);
    }

    void trwake_part(long long k) {                                   // samples, dipole sums -> doubles, two convolutions
        const elg_element& e = bl->e[k];
        count(); count(); count(); count();
        if (b) {
            launch_samples(k);
            dipole_finalize(e.nb);
            for (int plane = 0; plane < 2; plane++) {
                ConvArgs<double> cv;
                cv.counts = b->D + (size_t)plane * e.nb; cv.W = b->W; cv.st = b->st; cv.nb = e.nb; cv.q = b->q_macro;
                cv.V = b->Vt + (size_t)plane * e.nb;
                ProfScope ps(b, ELG_K_CONV);
                launch_k(conv_kernel<double>, (e.nb + kWarps - 1) / kWarps, kBlock, 0, b->stream, cv);
            }
            check(cudaGetLastError(), "conv_kernel launch");
            if (o && o->V_out && o->V_written + 4LL * e.nb <= o->V_capacity) {
                check(cudaMemcpyAsync(o->V_out + o->V_written, b->D, (size_t)e.nb * 16, cudaMemcpyDeviceToHost, b->stream), "D D2H");
                check(cudaMemcpyAsync(o->V_out + o->V_written + 2LL * e.nb, b->Vt, (size_t)e.nb * 16, cudaMemcpyDeviceToHost, b->stream), "Vt D2H");
            }
        }
        if (o) o->V_written += 4LL * e.nb;
        queue_tkick(e.nb, e.interp);
    }

    void stage_out_hist(int nb) {
        if (!o) return;
        if (o->window_out && o->window_written < o->window_capacity)
            check(cudaMemcpyAsync(o->window_out + 3 * o->window_written, b->st->win, 24, cudaMemcpyDeviceToHost, b->stream), "window D2H");
        o->window_written++;
        if (o->hist_out && o->hist_written + nb <= o->hist_capacity)
            check(cudaMemcpyAsync(o->hist_out + o->hist_written, b->counts, (size_t)nb * 4, cudaMemcpyDeviceToHost, b->stream), "hist D2H");
        o->hist_written += nb;
    }

    void run_turn(long long turn, long long k_begin = 0) {
        const long long ne = (long long)bl->e.size();
        const int mom = o ? o->moments_every : ELG_MOM_NONE;
        for (long long k = k_begin; k < ne && ok(); k++) {
            if (skip_next) { skip_next = false; continue; }           // TRWAKE merged into the preceding WAKE
            const elg_element& e = bl->e[k];
            const double s_here = bl->ring ? std::fma((double)turn, bl->length, bl->s_design[k]) : bl->s_design[k];   // G8
            bool recorded = false;
            HostOp op{};
            switch (e.type) {
                case ELG_DRIFT: op.type = OP_DRIFT; op.coef[0] = e.L; push(op); break;
                case ELG_MATRIX: push_matrix(e); break;
                case ELG_MATRIX2: case ELG_MATRIX3: push_higher_order(e); break;
                case ELG_RFKICK:
                    if (e.fiducial) {                                        // G36: needs the particles in memory
                        flush(AP_NONE, 0, 0, 0, false);
                        count();
                        if (b && ok()) {
                            ProfScope ps(b, ELG_K_MOMENTS);
                            launch_k(fiducial_kernel, b->grid_mom, kBlock, 0, b->stream, b->coord(b->cur_buf, 4), b->st, b->cur_slot, s_here);
                            check(cudaGetLastError(), "fiducial_kernel launch");
                        }
                        op.coef[5] = 1.0;
                    }
                    op.type = OP_RFKICK;
                    op.coef[0] = e.V * (b ? b->inv_E : 0.0); op.coef[1] = kTwoPi * e.f; op.coef[2] = e.phi;
                    op.coef[3] = s_here; op.coef[4] = b ? b->inv_bc : 0.0;
                    push(op);
                    break;
                case ELG_RCOL: case ELG_ECOL: {
                    const bool rect = e.type == ELG_RCOL;                    // ECOL carries 1/a, 1/b (G17)
                    const int ap = rect ? AP_RCOL : AP_ECOL;
                    const double px = rect ? e.ax : 1.0 / e.ax, py = rect ? e.ay : 1.0 / e.ay;
                    if (mom == ELG_MOM_ELEMENT) { moments_record(ap, px, py, (turn << 32) | k, next_is_hist(k, ne)); recorded = true; }
                    else flush(ap, px, py, (turn << 32) | k, next_is_hist(k, ne));
                    break;
                }
                case ELG_WAKE: case ELG_HISTO: case ELG_TRWAKE: wake_or_histo(k, s_here); break;
            }
            if (mom == ELG_MOM_ELEMENT && !recorded) moments_record();                       // G26
        }
        if (mom == ELG_MOM_TURN) moments_record();
    }
    // leading elements of the beamline that are plain per-particle maps (no collective step, aperture or record):
    // they can run chunk by chunk while later chunks are still being uploaded
    long long map_prefix() const {
        const long long ne = (long long)bl->e.size();
        if (o && o->moments_every == ELG_MOM_ELEMENT) return 0;
        long long k = 0;
        for (; k < ne; k++) {
            const elg_element& e = bl->e[k];
            const bool map = e.type == ELG_DRIFT || e.type == ELG_MATRIX || e.type == ELG_MATRIX2 || e.type == ELG_MATRIX3 ||
                             (e.type == ELG_RFKICK && !e.fiducial);
            if (!map) break;
        }
        return k;
    }

    // the map prefix of one turn on particles [lo, hi); the pending list is flushed with the min/max epilogue the next
    // element wants (slot = chunk index)
    void run_prefix_on_range(long long turn, long long k_end, long long lo, long long hi, int slot) {
        range_lo = lo; range_hi = hi; mm_slot = slot;
        const long long ne = (long long)bl->e.size();
        run_turn_range(turn, 0, k_end);
        flush(AP_NONE, 0, 0, 0, next_is_hist(k_end - 1, ne));
        range_lo = 0; range_hi = -1; mm_slot = 0;
    }
    void run_turn_range(long long turn, long long k_begin, long long k_end) {       // maps only (no records)
        for (long long k = k_begin; k < k_end && ok(); k++) {
            const elg_element& e = bl->e[k];
            const double s_here = bl->ring ? std::fma((double)turn, bl->length, bl->s_design[k]) : bl->s_design[k];
            HostOp op{};
            switch (e.type) {
                case ELG_DRIFT: op.type = OP_DRIFT; op.coef[0] = e.L; push(op); break;
                case ELG_MATRIX: push_matrix(e); break;
                case ELG_MATRIX2: case ELG_MATRIX3: push_higher_order(e); break;
                case ELG_RFKICK:
                    op.type = OP_RFKICK;
                    op.coef[0] = e.V * b->inv_E; op.coef[1] = kTwoPi * e.f; op.coef[2] = e.phi;
                    op.coef[3] = s_here; op.coef[4] = b->inv_bc;
                    push(op);
                    break;
                default: break;
            }
        }
    }

    bool next_is_hist(long long k, long long ne) const {
        return (k + 1 < ne) && (bl->e[k + 1].type == ELG_WAKE || bl->e[k + 1].type == ELG_HISTO || bl->e[k + 1].type == ELG_TRWAKE);
    }
};

int32_t upload_tables(elg_bunch* b, const elg_beamline* bl) {
    if (b->table_serial == bl->serial) return ELG_OK;
    if (bl->table_total > b->table_cap) return fail(ELG_ECAPACITY, "elg_track: workspace was sized for smaller wake tables");
    for (size_t k = 0; k < bl->e.size(); k++)
        if (!bl->table[k].empty())
            ELG_CK(cudaMemcpyAsync(b->table + bl->table_off[k], bl->table[k].data(), bl->table[k].size() * 8,
                                   cudaMemcpyHostToDevice, b->stream));
    b->table_serial = bl->serial;
    return ELG_OK;
}

}  // namespace

extern "C" int64_t elg_beamline_launches_per_turn(const elg_beamline* bl, int32_t moments_every) {
    if (!bl) return -1;
    elg_track_opts o{};
    o.moments_every = moments_every;
    Tracker t{nullptr, bl, &o};
    t.run_turn(0);
    t.flush(AP_NONE, 0, 0, 0, false);
    return t.launches;
}

extern "C" int32_t elg_track(elg_bunch* b, const elg_beamline* bl, int64_t n_turns, elg_track_opts* o) {
    if (!b || !bl || n_turns < 0) return fail(ELG_EINVAL, "elg_track: bad arguments");
    if (o) { o->n_records = 0; o->hist_written = 0; o->V_written = 0; o->window_written = 0; }
    // The caller may CAPTURE this call into a CUDA graph (cudaStreamBeginCapture on the bunch's stream): nothing in it
    // synchronises or reads the device when no host output is asked for.  A replay repeats the launches with the
    // parameters of the capture, so it is valid from the bunch state the capture started from (typically a captured
    // copy of the particles + elg_bunch_rewind in front of it).  The compaction's tile status is cleared at the head of
    // the captured work and its epoch restarted, so that the words of an earlier replay never look current.
    {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        ELG_CK(cudaStreamIsCapturing(b->stream, &cs));
        if (cs != cudaStreamCaptureStatusNone) {
            if (o && (o->records || o->hist_out || o->V_out || o->window_out))
                return fail(ELG_ESTATE, "elg_track: host outputs cannot be captured into a CUDA graph");
            if (b->prof_on) return fail(ELG_ESTATE, "elg_track: per-kernel profiling cannot be captured into a CUDA graph");
            if (b->table_serial != bl->serial && bl->table_total > 0)
                return fail(ELG_ESTATE, "elg_track: run this beamline once before capturing it (wake tables are uploaded on first use)");
            ELG_CK(cudaMemsetAsync(b->tile_status, 0, (b->stride / kStatusTile + 2) * 8, b->stream));
            b->epoch = 0;
        }
    }
    { int32_t rc = upload_tables(b, bl); if (rc != ELG_OK) return rc; }
    Tracker t{b, bl, o};
    b->rec_count = 0;
    for (int64_t it = 0; it < n_turns && t.ok(); it++) {
        t.run_turn(b->turn);
        b->turn++;
    }
    t.flush(AP_NONE, 0, 0, 0, false);
    if (t.ok()) t.flush_records();
    if (o) o->n_records = t.rec_total;
    if (t.ok() && o && (o->records || o->hist_out || o->V_out || o->window_out)) {
        cudaError_t e = cudaStreamSynchronize(b->stream);
        if (e != cudaSuccess) return fail(ELG_ECUDA, std::string("cudaStreamSynchronize: ") + cudaGetErrorString(e));
    }
    return t.rc;
}

// elg_bunch_upload + elg_track in one call, with the upload pipelined against the tracking: the bunch is cut into
// n_chunks particle ranges, each range is copied on the library's own copy stream and, as soon as it has landed, the
// leading per-particle maps of the first turn (everything in front of the first collective element, aperture or
// record) run on it while the next ranges are still crossing PCIe.  Results are identical to upload followed by track.
extern "C" int32_t elg_upload_and_track(elg_bunch* b, const elg_beamline* bl, const double* const h_coords[6],
                                        const int64_t* h_ids, int64_t n_turns, elg_track_opts* o, int32_t n_chunks) {
    if (!b || !bl || !h_coords || n_turns < 0) return fail(ELG_EINVAL, "elg_upload_and_track: bad arguments");
    for (int c = 0; c < 6; c++) if (!h_coords[c]) return fail(ELG_EINVAL, "elg_upload_and_track: NULL coordinate array");
    {
        cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
        ELG_CK(cudaStreamIsCapturing(b->stream, &cs));
        if (cs != cudaStreamCaptureStatusNone)
            return fail(ELG_ESTATE, "elg_upload_and_track: cannot be captured into a CUDA graph (host copies on a second stream); capture elg_track");
    }
    Tracker probe{b, bl, o};
    const long long k_split = probe.map_prefix();
    if (n_turns < 1 || k_split == 0 || n_chunks <= 1 || b->n0 < 4 * 9216) {       // nothing to overlap
        int32_t rc = elg_bunch_upload(b, h_coords, h_ids);
        return rc != ELG_OK ? rc : elg_track(b, bl, n_turns, o);
    }
    if (o) { o->n_records = 0; o->hist_written = 0; o->V_written = 0; o->window_written = 0; }
    if (!b->copy_stream) {
        ELG_CK(cudaStreamCreateWithFlags(&b->copy_stream, cudaStreamNonBlocking));
        ELG_CK(cudaEventCreateWithFlags(&b->entry_ev, cudaEventDisableTiming));
    }
    if (n_chunks > 32) n_chunks = 32;                               // min/max partial slots: 32 chunks x 444 blocks <= kMmPartials
    while ((int)b->chunk_ev.size() < n_chunks) {
        cudaEvent_t e = nullptr;
        ELG_CK(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
        b->chunk_ev.push_back(e);
    }
    // the copies overwrite store 0: everything queued on the bunch's stream so far must be done with it
    ELG_CK(cudaEventRecord(b->entry_ev, b->stream));
    ELG_CK(cudaStreamWaitEvent(b->copy_stream, b->entry_ev, 0));
    if (h_ids) ELG_CK(cudaMemcpyAsync(b->ids(0), h_ids, b->n0 * 8, cudaMemcpyHostToDevice, b->stream));
    else {
        launch_k(iota_kernel, b->sms * 4, kBlock, 0, b->stream, b->ids(0), b->n0);
        g_launches++;
        ELG_CK(cudaGetLastError());
    }
    { int32_t rc = elg_bunch_rewind(b); if (rc != ELG_OK) return rc; }
    { int32_t rc = upload_tables(b, bl); if (rc != ELG_OK) return rc; }
    Tracker t{b, bl, o};
    b->rec_count = 0;
    const long long per = align_up((b->n0 + n_chunks - 1) / n_chunks, 9216);     // multiple of every chain tile size (512 ... 2304)
    int slot = 0;
    for (long long lo = 0; lo < b->n0 && t.ok(); lo += per, slot++) {
        const long long hi = lo + per < b->n0 ? lo + per : b->n0;
        for (int c = 0; c < 6; c++)
            ELG_CK(cudaMemcpyAsync(b->coord(0, c) + lo, h_coords[c] + lo, (size_t)(hi - lo) * 8, cudaMemcpyHostToDevice, b->copy_stream));
        ELG_CK(cudaEventRecord(b->chunk_ev[slot], b->copy_stream));
        ELG_CK(cudaStreamWaitEvent(b->stream, b->chunk_ev[slot], 0));
        t.run_prefix_on_range(b->turn, k_split, lo, hi, slot);
    }
    if (t.ok()) t.run_turn(b->turn, k_split);
    b->turn++;
    for (int64_t it = 1; it < n_turns && t.ok(); it++) {
        t.run_turn(b->turn);
        b->turn++;
    }
    t.flush(AP_NONE, 0, 0, 0, false);
    if (t.ok()) t.flush_records();
    if (o) o->n_records = t.rec_total;
    if (t.ok() && o && (o->records || o->hist_out || o->V_out || o->window_out)) {
        cudaError_t e = cudaStreamSynchronize(b->stream);
        if (e != cudaSuccess) return fail(ELG_ECUDA, std::string("cudaStreamSynchronize: ") + cudaGetErrorString(e));
    }
    return t.rc;
}

// ------------------------------------------------------------------------------------- CUDA-graph support
// The host keeps a mirror of what it needs to know about the device state without ever reading it (which store holds
// the live particles, which count slot is current, the compaction epoch, the turn number, the records in the device
// ring).  A graph replay advances the device exactly as the captured call did but not this mirror: the caller saves
// it after the capture and puts it back after every replay.
extern "C" int32_t elg_bunch_host_state_save(const elg_bunch* b, int64_t out[8]) {
    if (!b || !out) return fail(ELG_EINVAL, "elg_bunch_host_state_save: bad arguments");
    out[0] = b->cur_buf; out[1] = b->cur_slot; out[2] = (int64_t)b->epoch; out[3] = b->turn; out[4] = b->rec_count;
    out[5] = 0; out[6] = 0; out[7] = 0x656c67;                    // tag
    return ELG_OK;
}
extern "C" int32_t elg_bunch_host_state_restore(elg_bunch* b, const int64_t in[8]) {
    if (!b || !in || in[7] != 0x656c67 || (in[0] | 1) != 1 || (in[1] | 1) != 1 || in[2] < 0 || in[2] > 0x3fffffff || in[4] < 0 || in[4] > kRecCap)
        return fail(ELG_EINVAL, "elg_bunch_host_state_restore: not a state written by elg_bunch_host_state_save");
    b->cur_buf = (int)in[0]; b->cur_slot = (int)in[1]; b->epoch = (unsigned int)in[2]; b->turn = in[3]; b->rec_count = in[4];
    return ELG_OK;
}

// ------------------------------------------------------------------------------------- host readbacks
extern "C" int32_t elg_n_alive(elg_bunch* b, int64_t* n_alive) {
    if (!b || !n_alive) return fail(ELG_EINVAL, "elg_n_alive: bad arguments");
    long long n = 0;
    ELG_CK(cudaMemcpyAsync(&n, &b->st->n_alive[b->cur_slot], 8, cudaMemcpyDeviceToHost, b->stream));
    ELG_CK(cudaStreamSynchronize(b->stream));
    *n_alive = n;
    return ELG_OK;
}

extern "C" int32_t elg_moments(elg_bunch* b, int64_t* n_alive, double h_centroid[6], double h_sigma[36]) {
    if (!b) return fail(ELG_EINVAL, "elg_moments: NULL bunch");
    MomArgs m;
    for (int k = 0; k < 6; k++) m.src[k] = b->coord(b->cur_buf, k);
    m.st = b->st; m.cur = b->cur_slot; m.partial = b->mom_partial; m.prof_kind = -1;
    m.record = b->records + 43 * kRecCap;
    launch_k(moments_kernel, b->grid_mom, kBlock, 0, b->stream, m);
    g_launches++;
    ELG_CK(cudaGetLastError());
    double rec[43];
    ELG_CK(cudaMemcpyAsync(rec, m.record, sizeof rec, cudaMemcpyDeviceToHost, b->stream));
    ELG_CK(cudaStreamSynchronize(b->stream));
    if (n_alive) *n_alive = (int64_t)rec[0];
    if (rec[0] <= 0.0) return fail(ELG_ESTATE, "elg_moments: no live particles");
    if (h_centroid) std::memcpy(h_centroid, rec + 1, 6 * sizeof(double));
    if (h_sigma) std::memcpy(h_sigma, rec + 7, 36 * sizeof(double));
    return ELG_OK;
}

extern "C" int32_t elg_bunch_read(elg_bunch* b, double* const h_coords[6], int64_t* h_ids, int64_t cap) {
    if (!b) return fail(ELG_EINVAL, "elg_bunch_read: NULL bunch");
    int64_t n = 0;
    { int32_t rc = elg_n_alive(b, &n); if (rc != ELG_OK) return rc; }
    if (cap < n) return fail(ELG_ECAPACITY, "elg_bunch_read: capacity smaller than n_alive");
    if (n > 0) {
        for (int c = 0; c < 6; c++)
            if (h_coords && h_coords[c])
                ELG_CK(cudaMemcpyAsync(h_coords[c], b->coord(b->cur_buf, c), n * 8, cudaMemcpyDeviceToHost, b->stream));
        if (h_ids) ELG_CK(cudaMemcpyAsync(h_ids, b->ids(b->cur_buf), n * 8, cudaMemcpyDeviceToHost, b->stream));
        ELG_CK(cudaStreamSynchronize(b->stream));
    }
    return ELG_OK;
}

extern "C" int32_t elg_lost(elg_bunch* b, int64_t* n_lost, int64_t cap, int64_t* h_ids, int32_t* h_turn, int32_t* h_elem,
                            double* h_coords6) {
    if (!b || cap < 0) return fail(ELG_EINVAL, "elg_lost: bad arguments");
    long long nl = 0;
    ELG_CK(cudaMemcpyAsync(&nl, &b->st->n_lost[b->cur_slot], 8, cudaMemcpyDeviceToHost, b->stream));
    ELG_CK(cudaStreamSynchronize(b->stream));
    if (n_lost) *n_lost = nl;
    long long have = nl < b->lost_cap ? nl : b->lost_cap;           // records kept on the device
    long long m = have < cap ? have : cap;
    if (m > 0) {
        if (h_ids) ELG_CK(cudaMemcpyAsync(h_ids, b->lost_id, m * 8, cudaMemcpyDeviceToHost, b->stream));
        std::vector<long long> te;
        if (h_turn || h_elem) {
            te.resize(m);
            ELG_CK(cudaMemcpyAsync(te.data(), b->lost_te, m * 8, cudaMemcpyDeviceToHost, b->stream));
        }
        std::vector<double> tmp;
        if (h_coords6) {
            tmp.resize(6 * m);
            for (int c = 0; c < 6; c++)
                ELG_CK(cudaMemcpyAsync(tmp.data() + c * m, b->lost_v + c * b->lost_cap, m * 8, cudaMemcpyDeviceToHost, b->stream));
        }
        ELG_CK(cudaStreamSynchronize(b->stream));
        for (long long j = 0; j < m; j++) {
            if (h_turn) h_turn[j] = (int32_t)(te[j] >> 32);
            if (h_elem) h_elem[j] = (int32_t)(te[j] & 0xffffffffLL);
            if (h_coords6) for (int c = 0; c < 6; c++) h_coords6[6 * j + c] = tmp[c * m + j];   // layout only
        }
    }
    if (cap < nl) return fail(ELG_ECAPACITY, "elg_lost: more lost particles than capacity");
    return ELG_OK;
}

extern "C" int32_t elg_bunch_device_array(elg_bunch* b, int32_t c, void** d_ptr) {
    if (!b || !d_ptr || c < 0 || c > 6) return fail(ELG_EINVAL, "elg_bunch_device_array: bad arguments");
    *d_ptr = (c < 6) ? (void*)b->coord(b->cur_buf, c) : (void*)b->ids(b->cur_buf);
    return ELG_OK;
}

// ------------------------------------------------------------------------------------- test hooks
// The hooks below run ONE stage of elg_track on the particles currently in the bunch (the caller uploads the oracle's
// input of that stage first), through the same planner code (Tracker) and hence the same kernels and launch
// configurations as tracking itself.
namespace {
elg_element hook_window_element(double dt, int32_t nb) {
    elg_element e{};
    e.type = ELG_HISTO; e.nb = nb; e.window = ELG_WIN_EXPLICIT; e.t_lo_rel = 0.0; e.dt = dt;   // t_lo = t_design + 0
    return e;
}
int32_t hook_check(const elg_bunch* b, double dt, int32_t nb, const char* who) {
    if (!b || nb < 2 || !(dt > 0.0)) return fail(ELG_EINVAL, std::string(who) + ": bad arguments");
    if (nb > b->nb_cap) return fail(ELG_ECAPACITY, std::string(who) + ": workspace was sized for fewer bins");
    return ELG_OK;
}
}  // namespace

extern "C" int32_t elg_dbg_histogram(elg_bunch* b, double t_lo, double dt, int32_t nb, uint32_t* d_counts) {
    { int32_t rc = hook_check(b, dt, nb, "elg_dbg_histogram"); if (rc != ELG_OK) return rc; }
    if (!d_counts) return fail(ELG_EINVAL, "elg_dbg_histogram: NULL output");
    Tracker t{b, nullptr, nullptr};
    t.prepare_hist(hook_window_element(dt, nb), t_lo, false);
    if (!t.ok()) return t.rc;
    ELG_CK(cudaMemcpyAsync(d_counts, b->counts, (size_t)nb * 4, cudaMemcpyDeviceToDevice, b->stream));
    return ELG_OK;
}

extern "C" int32_t elg_dbg_dipole_histogram(elg_bunch* b, double t_lo, double dt, int32_t nb, uint32_t* d_counts, double* d_D) {
    { int32_t rc = hook_check(b, dt, nb, "elg_dbg_dipole_histogram"); if (rc != ELG_OK) return rc; }
    if (!d_counts || !d_D) return fail(ELG_EINVAL, "elg_dbg_dipole_histogram: NULL output");
    Tracker t{b, nullptr, nullptr};
    t.prepare_hist(hook_window_element(dt, nb), t_lo, true);
    if (!t.ok()) return t.rc;
    t.dipole_finalize(nb);
    if (!t.ok()) return t.rc;
    ELG_CK(cudaMemcpyAsync(d_counts, b->counts, (size_t)nb * 4, cudaMemcpyDeviceToDevice, b->stream));
    ELG_CK(cudaMemcpyAsync(d_D, b->D, (size_t)nb * 16, cudaMemcpyDeviceToDevice, b->stream));
    return ELG_OK;
}

// the wake kick exactly as tracking applies it: OP_KICK / OP_TKICK as a fused run of one op, behind the min/max
// epilogue and the window kernel that set the device-resident window
extern "C" int32_t elg_dbg_kick(elg_bunch* b, double t_lo, double dt, int32_t nb, const double* d_V, int32_t interp) {
    { int32_t rc = hook_check(b, dt, nb, "elg_dbg_kick"); if (rc != ELG_OK) return rc; }
    if (!d_V) return fail(ELG_EINVAL, "elg_dbg_kick: NULL V");
    Tracker t{b, nullptr, nullptr};
    t.flush(AP_NONE, 0, 0, 0, true);
    t.launch_window(hook_window_element(dt, nb), t_lo, false);
    if (!t.ok()) return t.rc;
    ELG_CK(cudaMemcpyAsync(b->V, d_V, (size_t)nb * 8, cudaMemcpyDeviceToDevice, b->stream));
    t.queue_kick(nb, interp);
    t.flush(AP_NONE, 0, 0, 0, false);
    return t.rc;
}

extern "C" int32_t elg_dbg_tkick(elg_bunch* b, double t_lo, double dt, int32_t nb, const double* d_Vx, const double* d_Vy,
                                 int32_t interp) {
    { int32_t rc = hook_check(b, dt, nb, "elg_dbg_tkick"); if (rc != ELG_OK) return rc; }
    if (!d_Vx || !d_Vy) return fail(ELG_EINVAL, "elg_dbg_tkick: NULL V");
    Tracker t{b, nullptr, nullptr};
    t.flush(AP_NONE, 0, 0, 0, true);
    t.launch_window(hook_window_element(dt, nb), t_lo, false);
    if (!t.ok()) return t.rc;
    ELG_CK(cudaMemcpyAsync(b->Vt, d_Vx, (size_t)nb * 8, cudaMemcpyDeviceToDevice, b->stream));
    ELG_CK(cudaMemcpyAsync(b->Vt + nb, d_Vy, (size_t)nb * 8, cudaMemcpyDeviceToDevice, b->stream));
    t.queue_tkick(nb, interp);
    t.flush(AP_NONE, 0, 0, 0, false);
    return t.rc;
}

// aperture + stable compaction alone: a run of zero maps ending in the aperture (PAPER.md:141 loss contract)
extern "C" int32_t elg_dbg_compact(elg_bunch* b, int32_t type, double ax, double ay) {
    if (!b || (type != ELG_RCOL && type != ELG_ECOL) || !(ax > 0.0) || !(ay > 0.0))
        return fail(ELG_EINVAL, "elg_dbg_compact: bad arguments");
    Tracker t{b, nullptr, nullptr};
    const bool rect = type == ELG_RCOL;
    t.flush(rect ? AP_RCOL : AP_ECOL, rect ? ax : 1.0 / ax, rect ? ay : 1.0 / ay, (b->turn << 32), false);
    return t.rc;
}

extern "C" int32_t elg_dbg_wake_samples(int32_t kind, int32_t nb, double dt, double f, double Q, double Rs,
                                        const double* d_table, int64_t n_table, double dt_table, double* d_W, void* stream) {
    if (nb < 1 || !d_W || !(dt > 0.0)) return fail(ELG_EINVAL, "elg_dbg_wake_samples: bad arguments");
    WakeArgs wa{};
    wa.st = nullptr; wa.dt_fixed = dt; wa.kind = kind; wa.nb = nb;
    if (kind == ELG_WAKE_RESONATOR) {
        if (!(Q > 0.5)) return fail(ELG_EINVAL, "elg_dbg_wake_samples: Q <= 1/2");
        const double wr = kTwoPi * f;
        wa.kloss = wr * Rs / (2.0 * Q);
        wa.alpha = wr / (2.0 * Q);
        wa.wbar = std::sqrt(wr * wr - wa.alpha * wa.alpha);
        wa.ratio = wa.alpha / wa.wbar;
    } else if (kind == ELG_WAKE_TABLE) {
        if (!d_table || n_table < 1 || !(dt_table > 0.0)) return fail(ELG_EINVAL, "elg_dbg_wake_samples: bad table");
    } else return fail(ELG_EINVAL, "elg_dbg_wake_samples: bad kind");
    wa.table = d_table; wa.n_table = n_table; wa.dt_table = dt_table; wa.W = d_W;
    launch_k(wake_samples_kernel, (nb + kBlock - 1) / kBlock, kBlock, 0, (cudaStream_t)stream, wa);
    g_launches++;
    ELG_CK(cudaGetLastError());
    return ELG_OK;
}

extern "C" int32_t elg_dbg_convolve(const uint32_t* d_counts, const double* d_W, int32_t nb, double q, double* d_V,
                                    void* stream) {
    if (nb < 1 || !d_counts || !d_W || !d_V) return fail(ELG_EINVAL, "elg_dbg_convolve: bad arguments");
    ConvArgs<unsigned int> cv;
    cv.counts = d_counts; cv.W = d_W; cv.st = nullptr; cv.nb = nb; cv.q = q; cv.V = d_V;
    launch_k(conv_kernel<unsigned int>, (nb + kWarps - 1) / kWarps, kBlock, 0, (cudaStream_t)stream, cv);
    g_launches++;
    ELG_CK(cudaGetLastError());
    return ELG_OK;
}

// =====================================================================================================
// elg_dipole_histogram_noalloc: the dipole histogram stage (TRWAKE, G32-G33) for callers that cannot allocate and have
// no workspace to lend (code under CUDA-graph capture, tight serving loops, harnesses that forbid cudaMalloc).  The
// scratch the stage needs -- a device state block and four 64-bit fixed-point accumulators per bin -- lives in a
// file-scope device array of fixed size, held by every GPU that loads the library until the process exits:
// 512 B + 32 B x kNoAllocMaxBins = 524 800 bytes.  The call allocates nothing (no cudaMalloc / cudaFree, no allocating
// library routine): it launches a prepare kernel (state, zeroed accumulators, zeroed output counts), tracking's own
// dipole_hist_kernel and dipole_finalize_kernel on the caller's stream.
// In HOST code the array's name is a host-side stand-in, not a device address: the address is asked for once per
// device, with that device current (cudaGetSymbolAddress), and handed to the kernels.
// All calls on a device share the array and it keeps the last call's contents: every call clears what must start at
// zero, and two calls that overlap on the GPU (different streams, no ordering between them) RACE on it.
// =====================================================================================================
namespace {
constexpr int kNoAllocMaxBins = 16384;
constexpr size_t kNoAllocStateBytes = 512;                               // >= sizeof(DevState)
constexpr size_t kNoAllocBytes = kNoAllocStateBytes + (size_t)kNoAllocMaxBins * 4 * sizeof(unsigned long long);
static_assert(sizeof(DevState) <= kNoAllocStateBytes, "state block of the static scratch");
}  // namespace
static __device__ __align__(256) unsigned char g_noalloc_scratch[kNoAllocBytes];

namespace {
// fills the state block the histogram kernel reads (n, EXPLICIT window, whole bin range) and clears what accumulates
__global__ void __launch_bounds__(kBlock) noalloc_prepare_kernel(unsigned char* scratch, long long n, double t_lo, double dt, int nb,
                                                                 unsigned int* counts) {
    DevState* st = reinterpret_cast<DevState*>(scratch);
    unsigned long long* dacc = reinterpret_cast<unsigned long long*>(scratch + kNoAllocStateBytes);
    const int stride = gridDim.x * kBlock;
    for (int i = blockIdx.x * kBlock + threadIdx.x; i < 4 * nb; i += stride) dacc[i] = 0ull;
    for (int i = blockIdx.x * kBlock + threadIdx.x; i < nb; i += stride) counts[i] = 0u;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        st->n_alive[0] = n; st->n_alive[1] = n; st->n_lost[0] = 0; st->n_lost[1] = 0;
        st->win[0] = t_lo; st->win[1] = dt; st->win[2] = 1.0 / dt; st->win[3] = 0.0;
        st->smin = 0.0; st->smax = 0.0;
        st->bin_lo = 0; st->bin_hi = nb - 1;
        st->zero_bits = 0;
    }
}

// device address of the scratch array on the CURRENT device, looked up once per device
int32_t noalloc_scratch(unsigned char** out) {
    constexpr int kMaxDevices = 64;
    static unsigned char* ptrs[kMaxDevices] = {nullptr};
    static std::atomic<int> have[kMaxDevices];
    int dev = 0;
    ELG_CK(cudaGetDevice(&dev));
    if (dev < 0 || dev >= kMaxDevices) return fail(ELG_EINVAL, "elg_dipole_histogram_noalloc: device index out of range");
    if (!have[dev].load(std::memory_order_acquire)) {
        unsigned char* p = nullptr;
        ELG_CK(cudaGetSymbolAddress((void**)&p, g_noalloc_scratch));
        if (!p) return fail(ELG_ECUDA, "elg_dipole_histogram_noalloc: cudaGetSymbolAddress returned NULL");
        ptrs[dev] = p;                                                   // (the same value from every thread that races here)
        have[dev].store(1, std::memory_order_release);
    }
    *out = ptrs[dev];
    return ELG_OK;
}
}  // namespace

extern "C" int32_t elg_noalloc_max_bins(void) { return kNoAllocMaxBins; }

extern "C" int32_t elg_dipole_histogram_noalloc(const double* d_s, const double* d_x, const double* d_y, int64_t n, double inv_bc,
                                                double t_lo, double dt, int32_t nb, uint32_t* d_counts, double* d_D, void* stream) {
    if (n < 0 || n >= (1LL << 31) || (n > 0 && (!d_s || !d_x || !d_y)) || !d_counts || !d_D || !(dt > 0.0) || !std::isfinite(t_lo) ||
        !std::isfinite(inv_bc))
        return fail(ELG_EINVAL, "elg_dipole_histogram_noalloc: bad arguments");
    if (nb < 2) return fail(ELG_EINVAL, "elg_dipole_histogram_noalloc: nb < 2");
    if (nb > kNoAllocMaxBins) {
        char buf[160];
        std::snprintf(buf, sizeof buf, "elg_dipole_histogram_noalloc: nb = %d exceeds the static scratch (at most %d bins)", (int)nb, kNoAllocMaxBins);
        return fail(ELG_ECAPACITY, buf);
    }
    if ((n > 0 && (((uintptr_t)d_s | (uintptr_t)d_x | (uintptr_t)d_y) & 15)) || ((uintptr_t)d_D & 7))
        return fail(ELG_EINVAL, "elg_dipole_histogram_noalloc: s, x, y must be 16-byte aligned");
    unsigned char* scratch = nullptr;
    { int32_t rc = noalloc_scratch(&scratch); if (rc != ELG_OK) return rc; }
    { int32_t rc = hist_setup_once(); if (rc != ELG_OK) return rc; }
    int sms = 0;
    { int32_t rc = device_sms(&sms); if (rc != ELG_OK) return rc; }
    cudaStream_t st = (cudaStream_t)stream;
    noalloc_prepare_kernel<<<(4 * nb + kBlock - 1) / kBlock, kBlock, 0, st>>>(scratch, (long long)n, t_lo, dt, nb, d_counts);
    g_launches++;
    ELG_CK(cudaGetLastError());
    DipoleArgs d;
    d.s = d_s; d.x = d_x; d.y = d_y;
    d.st = reinterpret_cast<DevState*>(scratch); d.prof_kind = -1; d.cur = 0; d.inv_bc = inv_bc; d.nb = nb;
    d.smem_bins = nb < kDipoleSmemBins ? (nb + 31) / 32 * 32 : kDipoleSmemBins;
    d.counts = d_counts;
    d.dacc = reinterpret_cast<unsigned long long*>(scratch + kNoAllocStateBytes);
    int occ = 0;
    ELG_CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, dipole_hist_kernel, kBlock, (size_t)d.smem_bins * 36));
    if (occ < 1) occ = 1;
    dipole_hist_kernel<<<occ * sms, kBlock, (size_t)d.smem_bins * 36, st>>>(d);
    g_launches++;
    ELG_CK(cudaGetLastError());
    dipole_finalize_kernel<<<(nb + kBlock - 1) / kBlock, kBlock, 0, st>>>(d.dacc, nb, d_D);
    g_launches++;
    ELG_CK(cudaGetLastError());
    return ELG_OK;
}
