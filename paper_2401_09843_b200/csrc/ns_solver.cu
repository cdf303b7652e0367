// ns_solver.cu -- host side of libns: the C ABI of include/ns.h, the solver handle, the workspace
// arena and the launch sequences (RHS pipeline a1..a7, SSP-RK3 driver).  Launches only; every
// arithmetic step of the path runs in the kernels of this directory.  No CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <limits>
#include <map>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/ns.h"
#include "kernels_misc.cuh"
#include "ns_internal.h"
#include "twiddles_host.h"

using namespace ns;

struct ns_solver {
    std::string err;
    long long launches = 0;
    virtual ~ns_solver() {}
    virtual int set_initial(const void* u, ns_memspace ms) = 0;
    virtual int set_spectral(const void* u, ns_memspace ms) = 0;
    virtual int get_spectral(void* u, ns_memspace ms) = 0;
    virtual int rhs(void* out, ns_memspace ms) = 0;
    virtual int step_uniform(double dt) = 0;
    virtual int step_cfl(double cfl, double t_end, double* dt_out) = 0;
    virtual int step_dts(const double* dt) = 0;
    virtual int advance(double cfl, double t_end, int max_steps, int* steps_done) = 0;
    virtual int max_velocity(double* out) = 0;
    virtual int get_fields(void* out, ns_memspace ms) = 0;
    virtual int energy_spectrum(double* E, int nbins, bool enstrophy) = 0;
    virtual int structure_function(double* S, int nl) = 0;
    virtual int structure_function_p(double p, double* S, int nl) = 0;
    virtual int ensemble_moments(void* mean, void* var, ns_memspace ms) = 0;
    virtual double time(int sample) = 0;
    virtual long long device_bytes() const = 0;
    virtual int padded_size() const = 0;
    virtual int transform_grid() const = 0;
    virtual int time_transform(int reps, double* ms) = 0;
    virtual int profile(int enable) = 0;
    virtual int profile_read(double* ms, long long* cnt) = 0;
};

static thread_local std::string g_create_error;

namespace {

double dissipation_rate(const ns_params& p, int N, double k2) {
    if (k2 <= 0.0) return 0.0;
    double d = p.nu * k2;
    if (p.eps != 0.0) {
        const double kabs = std::sqrt(k2);
        const double mN = p.m_cut < 0.0 ? std::sqrt((double)N) : p.m_cut;
        const double qe = p.q_exp < 0.0 ? (2.0 * p.s - 1.0) * 2.0 : p.q_exp;
        if (kabs > mN) {
            const double Q = p.q_sharp ? 1.0 : 1.0 - std::pow(mN / kabs, qe);
            d += p.eps / std::pow((double)N, 2.0 * p.s - 1.0) * std::pow(k2, p.s) * Q;
        }
    }
    return d;
}

// Optional per-pass timing with CUDA events on the solver's stream (ns_profile / ns_profile_read).
// Passes: 0 a1 col_inv_x, 1 a2 col_inv_y, 2 a3 z_inv_prod, 3 a4 z_fwd, 4 a5 col_fwd_y, 5 a6 col_fwd_x,
//         6 a7 spectral, 7 other (dt bookkeeping).  An event is recorded at the start of every pass.
struct PassProfiler {
    static constexpr int NPASS = 8;
    static constexpr size_t MAX_EVENTS = 1 << 16;
    bool on = false;
    std::vector<cudaEvent_t> ev;
    std::vector<int> tag;
    size_t used = 0;
    double ms[NPASS] = {0};
    long long cnt[NPASS] = {0};
    ~PassProfiler() {
        for (cudaEvent_t e : ev) cudaEventDestroy(e);
    }
    void reset() {
        used = 0;
        for (int i = 0; i < NPASS; ++i) { ms[i] = 0; cnt[i] = 0; }
    }
    void reserve(size_t n) {   // events are created when profiling is switched on, not inside a timed loop
        while (ev.size() < n) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return;
            ev.push_back(e);
            tag.push_back(-1);
        }
    }
    void tick(int pass, cudaStream_t st) {  // pass < 0: end marker
        if (!on || used >= MAX_EVENTS) return;
        if (used == ev.size()) {
            cudaEvent_t e;
            if (cudaEventCreate(&e) != cudaSuccess) return;
            ev.push_back(e);
            tag.push_back(-1);
        }
        tag[used] = pass;
        cudaEventRecord(ev[used], st);
        ++used;
    }
    void collect() {  // stream must be synchronised
        for (size_t i = 0; i + 1 < used; ++i) {
            if (tag[i] < 0) continue;
            float t = 0;
            if (cudaEventElapsedTime(&t, ev[i], ev[i + 1]) == cudaSuccess) {
                ms[tag[i]] += t;
                cnt[tag[i]] += 1;
            }
        }
        used = 0;
    }
};

template <typename T>
class Solver final : public ns_solver {
public:
    int N, L, M, H, batch;   // N = the transform grid (N/2 a supported length), M = 3N/2 its padded grid
    int Nu;                  // the user's grid (public arrays, truncation set K_Nu, dx, eps_N, m_N); Nu <= N, see ns_create
    cx<T>* gNu = nullptr;    // exp(2 pi i j / Nu), j < Nu (unpadded transforms on the user's grid)
    int device = 0, num_sms = 0;   // the device the handle was created on (no process-wide caches)
    ns_params prm;
    cudaStream_t st;
    bool has_state = false;
    // arena
    unsigned char* arena = nullptr;
    size_t arena_bytes = 0;
    cx<T>*U = nullptr, *V = nullptr, *X = nullptr, *Y = nullptr, *Z = nullptr;
    cx<T>* twbase = nullptr;  // twiddle-table block (twiddles_host.h)
    T* dtab = nullptr;
    double *dt_dev = nullptr, *t_dev = nullptr, *scal_dev = nullptr, *red_dev = nullptr;
    unsigned long long* umax2 = nullptr;
    int* bad_dev = nullptr;   // per-sample flag: non-finite state seen (kernels_misc.cuh)
    size_t nS, nX, nY, nZ;  // complex element counts of state, X, Y, Z
    long XS = 0;            // pitch of one px row of X (a1 out / a5 out), complex elements
    size_t red_count;
    PassProfiler prof;
    Solver(int Nu_, int N_, int batch_, const ns_params& p, cudaStream_t s)
        : N(N_), L(N_ / 2), M(3 * N_ / 2), H(N_ / 2), batch(batch_), Nu(Nu_), prm(p), st(s) {}
    ~Solver() override {
        if (arena) cudaFree(arena);
    }

    int fail(int code, const std::string& msg) {
        err = msg;
        return code;
    }
    int cuda_fail(cudaError_t e, const char* where) {
        err = std::string(where) + ": " + cudaGetErrorString(e);
        return NS_ERR_CUDA;
    }
#define NS_CK(call)                                           \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)
#define NS_LAUNCHED(name)                                      \
    do {                                                       \
        ++launches;                                            \
        cudaError_t e__ = cudaGetLastError();                  \
        if (e__ != cudaSuccess) return cuda_fail(e__, name);   \
    } while (0)

    // Reads the per-sample non-finite flags (the stream is synchronised by the copy) and reports the first marked sample.
    int check_finite() {
        std::vector<int> bad((size_t)batch);
        NS_CK(cudaMemcpyAsync(bad.data(), bad_dev, (size_t)batch * sizeof(int), cudaMemcpyDeviceToHost, st));
        NS_CK(cudaStreamSynchronize(st));
        for (int b = 0; b < batch; ++b)
            if (bad[b]) {
                char buf[160];
                snprintf(buf, sizeof buf, "sample %d: the velocity field is not finite (NaN or inf); the sample is frozen", b);
                return fail(NS_ERR_NONFINITE, buf);
            }
        return NS_OK;
    }

    Twiddles<T> tw() const { return make_twiddles<T>(twbase, L); }
    static unsigned blocks_for(long total, int threads) { return (unsigned)((total + threads - 1) / threads); }

    int init() {
        NS_CK(cudaGetDevice(&device));
        NS_CK(cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, device));
        const size_t b = (size_t)batch;
        nS = b * 3 * N * N * H;
        // Workspaces shared by all passes: X <- a1 out / a5 out / unpadded-FFT cube / R,
        // Y <- a2 out / a6 out (B_hat) / host staging, Z <- fused-z out.
        XS = (long)N * H;                                 // row (px) pitch of the X workspace (padding it was measured: no gain)
        nX = b * NS_NFLUX * (size_t)M * XS;               // A1b; >= A1u (3 M N H), W (3 N^3 = 6 N^2 H), R (3 N^2 H)
        nY = b * 3 * (size_t)M * M * H;                   // A2u; >= Bh (5 N^2 H), public / physical staging
        nZ = b * NS_NFLUX * (size_t)M * M * H;            // A2b
        const size_t pub = b * 3 * (size_t)Nu * Nu * (Nu / 2 + 1);
        if (nY < pub) nY = pub;
        const size_t ndt = (size_t)3 * L * L + 1;
        red_count = b * (size_t)(4096 > 3 * N ? 4096 : 3 * N);
        auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
        size_t off = 0;
        auto take = [&](size_t bytes) { size_t o = off; off += al(bytes); return o; };
        const size_t oU = take(nS * sizeof(cx<T>)), oV = take(nS * sizeof(cx<T>));
        const size_t oX = take(nX * sizeof(cx<T>)), oY = take(nY * sizeof(cx<T>)), oZ = take(nZ * sizeof(cx<T>));
        const size_t otw = take(twiddle_table_len(L) * sizeof(cx<T>));
        const size_t ogu = take((size_t)Nu * sizeof(cx<T>));
        const size_t oD = take(ndt * sizeof(T));
        const size_t odt = take(b * sizeof(double)), ot = take(b * sizeof(double)), osc = take(b * sizeof(double));
        const size_t oum = take(b * sizeof(unsigned long long));
        const size_t obad = take(b * sizeof(int));
        const size_t ored = take(red_count * sizeof(double));
        arena_bytes = off;
        cudaError_t e = cudaMalloc(&arena, arena_bytes);
        if (e == cudaErrorMemoryAllocation) {
            cudaGetLastError();
            char buf[128];
            snprintf(buf, sizeof buf, "device allocation of %.2f GB failed", (double)arena_bytes / 1e9);
            return fail(NS_ERR_OOM, buf);
        }
        if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
        U = (cx<T>*)(arena + oU);
        V = (cx<T>*)(arena + oV);
        X = (cx<T>*)(arena + oX);
        Y = (cx<T>*)(arena + oY);
        Z = (cx<T>*)(arena + oZ);
        twbase = (cx<T>*)(arena + otw);
        gNu = (cx<T>*)(arena + ogu);
        dtab = (T*)(arena + oD);
        dt_dev = (double*)(arena + odt);
        t_dev = (double*)(arena + ot);
        scal_dev = (double*)(arena + osc);
        umax2 = (unsigned long long*)(arena + oum);
        bad_dev = (int*)(arena + obad);
        red_dev = (double*)(arena + ored);

        const std::vector<cx<T>> htw = build_twiddle_block<T>(L);
        std::vector<T> hd(ndt);
        for (size_t k2 = 0; k2 < ndt; ++k2) hd[k2] = (T)dissipation_rate(prm, Nu, (double)k2);   // eps_N, m_N of the USER's N
        std::vector<cx<T>> hgu((size_t)Nu);
        for (int j = 0; j < Nu; ++j) {
            const long double a = 6.283185307179586476925286766559005768L * (long double)j / (long double)Nu;
            hgu[(size_t)j].x = (T)cosl(a);
            hgu[(size_t)j].y = (T)sinl(a);
        }
        NS_CK(cudaMemcpyAsync(gNu, hgu.data(), hgu.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, st));
        NS_CK(cudaMemcpyAsync(twbase, htw.data(), htw.size() * sizeof(cx<T>), cudaMemcpyHostToDevice, st));
        NS_CK(cudaMemcpyAsync(dtab, hd.data(), hd.size() * sizeof(T), cudaMemcpyHostToDevice, st));
        NS_CK(cudaMemsetAsync(t_dev, 0, b * sizeof(double), st));
        NS_CK(cudaMemsetAsync(dt_dev, 0, b * sizeof(double), st));
        NS_CK(cudaMemsetAsync(bad_dev, 0, b * sizeof(int), st));
        NS_CK(cudaStreamSynchronize(st));
        return NS_OK;
    }

    long long device_bytes() const override { return (long long)arena_bytes; }

    // ---------------------------------------------------------------- RHS transform pipeline a1..a6
    // Every pass works on the samples [b0, b0 + nb) of the batch; workspaces are indexed by sample, so groups of samples use
    // disjoint ranges of X / Y / Z within a pass.  X holds 3 (a1 out) or 5 (a5 out) components per sample and Y 3 padded
    // (a2 out) or 5 truncated (a6 out).
    int pass_inverse(const cx<T>* Uin, int b0, int nb) {
        const long NH = (long)N * H, MH = (long)M * H;
        cudaError_t e;
        prof.tick(0, st);
        e = launch_col_inv<T>(st, num_sms, L, Uin + (size_t)b0 * 3 * N * NH, X + (size_t)b0 * 3 * M * XS, NH, (long)nb * 3, NH, XS,
                              (long)N * NH, (long)M * XS, tw());
        if (e != cudaSuccess) return cuda_fail(e, "a1 col_inv x");
        ++launches;
        prof.tick(1, st);
        e = launch_col_inv<T>(st, num_sms, L, X + (size_t)b0 * 3 * M * XS, Y + (size_t)b0 * 3 * M * MH, H, (long)nb * 3 * M, H, H, XS, MH, tw());
        if (e != cudaSuccess) return cuda_fail(e, "a2 col_inv y");
        ++launches;
        return NS_OK;
    }
    int pass_z(cudaStream_t s, int sms, int b0, int nb, bool want_umax) {
        const long MH = (long)M * H;
        prof.tick(2, s);
        cudaError_t e = launch_z_fused<T>(s, sms, L, Y + (size_t)b0 * 3 * M * MH, Z + (size_t)b0 * NS_NFLUX * M * MH, (long)M * M, nb,
                                          want_umax ? umax2 + b0 : nullptr, tw());
        if (e != cudaSuccess) return cuda_fail(e, "a3+a4 z_fused");
        ++launches;
        return NS_OK;
    }
    int pass_forward(int b0, int nb) {
        const long NH = (long)N * H, MH = (long)M * H;
        cudaError_t e;
        prof.tick(4, st);
        e = launch_col_fwd<T>(st, num_sms, L, Z + (size_t)b0 * NS_NFLUX * M * MH, X + (size_t)b0 * NS_NFLUX * M * XS, H,
                              (long)nb * NS_NFLUX * M, H, H, MH, XS, (T)1, tw());
        if (e != cudaSuccess) return cuda_fail(e, "a5 col_fwd y");
        ++launches;
        prof.tick(5, st);
        e = launch_col_fwd<T>(st, num_sms, L, X + (size_t)b0 * NS_NFLUX * M * XS, Y + (size_t)b0 * NS_NFLUX * N * NH, NH, (long)nb * NS_NFLUX,
                              XS, NH, (long)M * XS, (long)N * NH, (T)1, tw());
        if (e != cudaSuccess) return cuda_fail(e, "a6 col_fwd x");
        ++launches;
        prof.tick(7, st);
        return NS_OK;
    }

    // Uin (internal layout) -> Y = Th [b][5][N][N][H] (unnormalised transforms of the trace-free flux), all samples, one stream
    int transform(const cx<T>* Uin, bool want_umax, int upto = 6) {
        int rc;
        if ((rc = pass_inverse(Uin, 0, batch)) != NS_OK) return rc;
        if ((rc = pass_z(st, num_sms, 0, batch, want_umax)) != NS_OK) return rc;
        if (upto <= 3) { prof.tick(-1, st); return NS_OK; }
        return pass_forward(0, batch);
    }

    int spectral(const cx<T>* Us, const cx<T>* Un, cx<T>* out, double alpha, double beta, double gamma, int mode, int b0 = 0, int nb = -1) {
        if (nb < 0) nb = batch;
        const long plane = (long)N * N * H, total = (long)nb * plane;
        const T scale = (T)(1.0 / ((double)M * M * M * z_fused_output_scale(L)));
        prof.tick(6, st);
        spectral_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(Y + (size_t)b0 * NS_NFLUX * plane, Us + (size_t)b0 * 3 * plane,
                                                                    Un ? Un + (size_t)b0 * 3 * plane : nullptr, out + (size_t)b0 * 3 * plane, N,
                                                                    Nu / 2, total, dtab, scale, (T)alpha, (T)beta, (T)gamma, dt_dev + b0, mode, N, 0);
        NS_LAUNCHED("a7 spectral_kernel");
        prof.tick(-1, st);
        return NS_OK;
    }

    // One RK stage = transform + tail (time-step bookkeeping in stage 1, then a7).  A two-stream variant that ran the z kernel of
    // one group of samples beside the column passes of the others was measured and gained nothing (profiles/r02_experiments.md).
    template <typename Tail>
    int stage(const cx<T>* Uin, bool want_umax, Tail tail) {
        int rc = transform(Uin, want_umax);
        if (rc != NS_OK) return rc;
        return tail(0, batch);
    }

    // dt_dev / t_dev must have been set before the first spectral() of the step (stream order)
    enum DtMode { DT_UNIFORM, DT_ARRAY, DT_CFL };
    int rk3(DtMode mode, double dt, const double* dts_host, double cfl, double t_end) {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        int rc;
        // max|u|^2 is a free by-product of a3 in stage 1; besides the CFL step it is what detects a non-finite state
        NS_CK(cudaMemsetAsync(umax2, 0, (size_t)batch * sizeof(unsigned long long), st));
        if (mode == DT_ARRAY) NS_CK(cudaMemcpyAsync(scal_dev, dts_host, (size_t)batch * sizeof(double), cudaMemcpyHostToDevice, st));
        // eq. (2.6): u1 = u + dt R(u)
        rc = stage(U, true, [&](int b0, int nb) -> int {
            const unsigned gb = blocks_for(nb, 128);
            if (mode == DT_UNIFORM) {
                set_dt_uniform_kernel<<<gb, 128, 0, st>>>(dt_dev + b0, t_dev + b0, dt, umax2 + b0, bad_dev + b0, nb);
                NS_LAUNCHED("set_dt_uniform");
            } else if (mode == DT_ARRAY) {
                set_dt_array_kernel<<<gb, 128, 0, st>>>(dt_dev + b0, t_dev + b0, scal_dev + b0, umax2 + b0, bad_dev + b0, nb);
                NS_LAUNCHED("set_dt_array");
            } else {
                cfl_finalize_kernel<<<gb, 128, 0, st>>>(dt_dev + b0, t_dev + b0, umax2 + b0, bad_dev + b0, cfl, 2.0 * 3.14159265358979323846 / Nu,
                                                        t_end, nb);
                NS_LAUNCHED("cfl_finalize");
            }
            return spectral(U, nullptr, V, 0.0, 1.0, 1.0, 1, b0, nb);
        });
        if (rc != NS_OK) return rc;
        // u2 = 3/4 u + 1/4 u1 + 1/4 dt R(u1)
        rc = stage(V, false, [&](int b0, int nb) -> int { return spectral(V, U, V, 0.75, 0.25, 0.25, 1, b0, nb); });
        if (rc != NS_OK) return rc;
        // u+ = 1/3 u + 2/3 u2 + 2/3 dt R(u2)
        return stage(V, false, [&](int b0, int nb) -> int { return spectral(V, U, U, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, 1, b0, nb); });
    }

    int step_uniform(double dt) override {
        if (!(dt == dt) || std::isinf(dt)) return fail(NS_ERR_INVALID_ARG, "dt must be finite");
        return rk3(DT_UNIFORM, dt, nullptr, 0, 0);
    }
    int step_dts(const double* dts) override {
        if (!dts) return fail(NS_ERR_INVALID_ARG, "dt array is NULL");
        int rc = rk3(DT_ARRAY, 0, dts, 0, 0);
        if (rc != NS_OK) return rc;
        return check_finite();  // synchronises: dts is caller memory, do not return before it was read
    }
    int step_cfl(double cfl, double t_end, double* dt_out) override {
        if (!(cfl > 0.0)) return fail(NS_ERR_INVALID_ARG, "cfl must be positive");
        int rc = rk3(DT_CFL, 0, nullptr, cfl, t_end);
        if (rc != NS_OK) return rc;
        if (dt_out) {
            NS_CK(cudaMemcpyAsync(dt_out, dt_dev, (size_t)batch * sizeof(double), cudaMemcpyDeviceToHost, st));
            return check_finite();
        }
        return NS_OK;
    }

    int advance(double cfl, double t_end, int max_steps, int* steps_done) override {
        if (!(cfl > 0.0) || max_steps < 0 || !(t_end == t_end)) return fail(NS_ERR_INVALID_ARG, "need cfl > 0, max_steps >= 0, finite t_end");
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        std::vector<double> th((size_t)batch);
        int n = 0;
        while (n < max_steps) {
            NS_CK(cudaMemcpyAsync(th.data(), t_dev, (size_t)batch * sizeof(double), cudaMemcpyDeviceToHost, st));
            int rcf = check_finite();   // a non-finite sample has dt = 0 for ever: stop instead of spinning to max_steps
            if (rcf != NS_OK) { if (steps_done) *steps_done = n; return rcf; }
            bool done = true;
            for (double tb : th) done = done && !(tb < t_end);
            if (done) break;
            const int burst = max_steps - n < 4 ? max_steps - n : 4;
            for (int i = 0; i < burst; ++i) {
                int rc = rk3(DT_CFL, 0, nullptr, cfl, t_end);
                if (rc != NS_OK) return rc;
            }
            n += burst;
        }
        if (steps_done) *steps_done = n;
        return NS_OK;
    }

    int max_velocity(double* out) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        NS_CK(cudaMemsetAsync(umax2, 0, (size_t)batch * sizeof(unsigned long long), st));
        int rc = transform(U, true, 3);
        if (rc != NS_OK) return rc;
        umax_read_kernel<<<blocks_for(batch, 128), 128, 0, st>>>(scal_dev, umax2, bad_dev, batch);
        NS_LAUNCHED("umax_read");
        NS_CK(cudaMemcpyAsync(out, scal_dev, (size_t)batch * sizeof(double), cudaMemcpyDeviceToHost, st));
        return check_finite();   // umax_out is filled either way (+inf / NaN for the failed sample)
    }

    int rhs(void* out, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        int rc = transform(U, false);
        if (rc != NS_OK) return rc;
        if ((rc = spectral(U, nullptr, X, 0, 0, 0, 0)) != NS_OK) return rc;  // R -> X (internal layout)
        return export_spectral(X, out, ms);
    }

    // internal [b*3][N][N][H] -> public layout in caller memory
    int export_spectral(const cx<T>* src, void* out, ns_memspace ms) {
        const long total_pub = (long)batch * 3 * Nu * Nu * (Nu / 2 + 1);
        cx<T>* dst = ms == NS_DEVICE ? (cx<T>*)out : Y;
        to_public_kernel<T><<<blocks_for(total_pub, 256), 256, 0, st>>>(src, dst, N, Nu, total_pub);
        NS_LAUNCHED("to_public");
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(out, Y, (size_t)total_pub * sizeof(cx<T>), cudaMemcpyDeviceToHost, st));
            NS_CK(cudaStreamSynchronize(st));
        }
        return NS_OK;
    }

    int get_spectral(void* out, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        return export_spectral(U, out, ms);
    }

    int set_spectral(const void* in, ns_memspace ms) override {
        if (!in) return fail(NS_ERR_INVALID_ARG, "input pointer is NULL");
        const long total_pub = (long)batch * 3 * Nu * Nu * (Nu / 2 + 1);
        const cx<T>* src = (const cx<T>*)in;
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(Y, in, (size_t)total_pub * sizeof(cx<T>), cudaMemcpyHostToDevice, st));
            src = Y;
        }
        const long total = (long)batch * 3 * N * N * H;
        to_internal_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(src, U, N, Nu, total);
        NS_LAUNCHED("to_internal");
        NS_CK(cudaMemsetAsync(bad_dev, 0, (size_t)batch * sizeof(int), st));
        if (ms == NS_HOST) NS_CK(cudaStreamSynchronize(st));  // caller buffer fully consumed
        has_state = true;
        return NS_OK;
    }

    // unpadded 3-D transform on the USER's grid (cubes of Nu^3 complex), in place: mixed radix when Nu = p 2^a with p in
    // {1, 3, 5, 7, 15} and Nu a multiple of 8, else the plain DFT
    int generic_fft3(cx<T>* W, long cubes, int sign) {
        int odd = Nu, log2m = 0;
        while (odd % 2 == 0) { odd /= 2; ++log2m; }
        const bool fast = (odd == 1 || odd == 3 || odd == 5 || odd == 7 || odd == 15) && Nu % 8 == 0;
        if (fast) {
            const long tiles = cubes * (long)Nu * Nu / 8;
            const size_t smem = (size_t)Nu * 9 * sizeof(cx<T>);
            if (smem > 48 * 1024)
                NS_CK(cudaFuncSetAttribute(generic_fft_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            for (int axis = 0; axis < 3; ++axis) {
                generic_fft_kernel<T><<<(unsigned)tiles, 256, smem, st>>>(W, Nu, log2m, odd, axis, sign, tiles, gNu, 3);
                NS_LAUNCHED("generic_fft");
            }
        } else {
            const long tiles = cubes * (((long)Nu * Nu + 7) / 8);
            const size_t smem = (size_t)2 * Nu * 9 * sizeof(cx<T>);
            if (smem > 48 * 1024)
                NS_CK(cudaFuncSetAttribute(dft_lines_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            for (int axis = 0; axis < 3; ++axis) {
                dft_lines_kernel<T><<<(unsigned)tiles, 256, smem, st>>>(W, Nu, axis, sign, tiles, gNu, 3);
                NS_LAUNCHED("dft_lines");
            }
        }
        return NS_OK;
    }

    int set_initial(const void* in, ns_memspace ms) override {
        if (!in) return fail(NS_ERR_INVALID_ARG, "input pointer is NULL");
        const long cubes = (long)batch * 3;
        const long total = cubes * Nu * Nu * Nu;
        const T* src = (const T*)in;
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(Y, in, (size_t)total * sizeof(T), cudaMemcpyHostToDevice, st));
            src = reinterpret_cast<const T*>(Y);
        }
        real_to_complex_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(src, X, total);
        NS_LAUNCHED("real_to_complex");
        int rc = generic_fft3(X, cubes, -1);
        if (rc != NS_OK) return rc;
        const long tot = (long)batch * N * N * H;
        init_project_kernel<T><<<blocks_for(tot, 256), 256, 0, st>>>(X, U, N, Nu, tot, (T)(1.0 / ((double)Nu * Nu * Nu)));
        NS_LAUNCHED("init_project");
        NS_CK(cudaMemsetAsync(t_dev, 0, (size_t)batch * sizeof(double), st));
        NS_CK(cudaMemsetAsync(bad_dev, 0, (size_t)batch * sizeof(int), st));
        if (ms == NS_HOST) NS_CK(cudaStreamSynchronize(st));
        has_state = true;
        return NS_OK;
    }

    int get_fields(void* out, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        const long cubes = (long)batch * 3;
        const long total = cubes * Nu * Nu * Nu;
        expand_hermitian_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(U, X, N, Nu, total);
        NS_LAUNCHED("expand_hermitian");
        int rc = generic_fft3(X, cubes, +1);
        if (rc != NS_OK) return rc;
        T* dst = ms == NS_DEVICE ? (T*)out : reinterpret_cast<T*>(Y);
        complex_to_real_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(X, dst, total);
        NS_LAUNCHED("complex_to_real");
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(out, dst, (size_t)total * sizeof(T), cudaMemcpyDeviceToHost, st));
            NS_CK(cudaStreamSynchronize(st));
        }
        return NS_OK;
    }

    int energy_spectrum(double* E, int nbins, bool enstrophy) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!E || nbins < 1 || nbins > 4096) return fail(NS_ERR_INVALID_ARG, "E is NULL or nbins not in [1, 4096]");
        NS_CK(cudaMemsetAsync(red_dev, 0, (size_t)batch * nbins * sizeof(double), st));
        const long plane = (long)N * N * H;
        unsigned chunks = blocks_for(plane, 256 * 16);
        if (chunks > 1024) chunks = 1024;
        if (enstrophy)
            energy_spectrum_kernel<T, true><<<dim3(chunks, batch), 256, (size_t)nbins * sizeof(double), st>>>(U, red_dev, N, nbins);
        else
            energy_spectrum_kernel<T, false><<<dim3(chunks, batch), 256, (size_t)nbins * sizeof(double), st>>>(U, red_dev, N, nbins);
        NS_LAUNCHED("energy_spectrum");
        NS_CK(cudaMemcpyAsync(E, red_dev, (size_t)batch * nbins * sizeof(double), cudaMemcpyDeviceToHost, st));
        NS_CK(cudaStreamSynchronize(st));
        return NS_OK;
    }

    int structure_function(double* S, int nl) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!S || nl < 1 || nl > Nu / 2) return fail(NS_ERR_INVALID_ARG, "S is NULL or nl not in [1, N/2]");
        NS_CK(cudaMemsetAsync(red_dev, 0, (size_t)batch * 3 * N * sizeof(double), st));
        const long plane = (long)N * N * H;
        unsigned chunks = blocks_for(plane, 256 * 16);
        if (chunks > 1024) chunks = 1024;
        sf_marginals_kernel<T><<<dim3(chunks, batch), 256, (size_t)3 * N * sizeof(double), st>>>(U, red_dev, N);
        NS_LAUNCHED("sf_marginals");
        double* out_dev = reinterpret_cast<double*>(Y);
        sf_finalize_kernel<<<batch, 128, 0, st>>>(red_dev, out_dev, N, Nu, nl);
        NS_LAUNCHED("sf_finalize");
        NS_CK(cudaMemcpyAsync(S, out_dev, (size_t)batch * nl * sizeof(double), cudaMemcpyDeviceToHost, st));
        NS_CK(cudaStreamSynchronize(st));
        return NS_OK;
    }

    int structure_function_p(double p, double* S, int nl) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!S || nl < 1 || nl > Nu / 2 || !(p > 0.0) || std::isinf(p)) return fail(NS_ERR_INVALID_ARG, "S is NULL, nl not in [1, N/2] or p not positive and finite");
        // physical fields on the N grid, as in get_fields: Hermitian expansion -> unpadded inverse FFT -> reals in Y
        const long cubes = (long)batch * 3;
        const long total = cubes * Nu * Nu * Nu;
        expand_hermitian_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(U, X, N, Nu, total);
        NS_LAUNCHED("expand_hermitian");
        int rc = generic_fft3(X, cubes, +1);
        if (rc != NS_OK) return rc;
        T* phys = reinterpret_cast<T*>(Y);
        complex_to_real_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(X, phys, total);
        NS_LAUNCHED("complex_to_real");
        NS_CK(cudaMemsetAsync(red_dev, 0, (size_t)batch * nl * sizeof(double), st));
        const long np = (long)Nu * Nu * Nu;
        unsigned chunks = blocks_for(np, 256 * 8);
        if (chunks > 592) chunks = 592;
        sf_p_kernel<T><<<dim3(chunks, nl, batch), 256, 0, st>>>(phys, red_dev, Nu, nl, p);
        NS_LAUNCHED("sf_p");
        scale_kernel<<<blocks_for((long)batch * nl, 128), 128, 0, st>>>(red_dev, 1.0 / (3.0 * (double)np), batch * nl);
        NS_LAUNCHED("scale");
        NS_CK(cudaMemcpyAsync(S, red_dev, (size_t)batch * nl * sizeof(double), cudaMemcpyDeviceToHost, st));
        NS_CK(cudaStreamSynchronize(st));
        return NS_OK;
    }

    int ensemble_moments(void* mean, void* var, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!mean && !var) return fail(NS_ERR_INVALID_ARG, "both output pointers are NULL");
        const long cubes = (long)batch * 3;
        const long total = cubes * Nu * Nu * Nu;
        expand_hermitian_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(U, X, N, Nu, total);
        NS_LAUNCHED("expand_hermitian");
        int rc = generic_fft3(X, cubes, +1);
        if (rc != NS_OK) return rc;
        T* phys = reinterpret_cast<T*>(Y);
        complex_to_real_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(X, phys, total);
        NS_LAUNCHED("complex_to_real");
        const long n = 3L * Nu * Nu * Nu;              // X is free again: mean | var staged there
        T* dmean = reinterpret_cast<T*>(X);
        T* dvar = dmean + n;
        ensemble_moments_kernel<T><<<blocks_for(n, 256), 256, 0, st>>>(phys, dmean, dvar, n, batch);
        NS_LAUNCHED("ensemble_moments");
        const cudaMemcpyKind kind = ms == NS_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
        if (mean) NS_CK(cudaMemcpyAsync(mean, dmean, (size_t)n * sizeof(T), kind, st));
        if (var) NS_CK(cudaMemcpyAsync(var, dvar, (size_t)n * sizeof(T), kind, st));
        if (ms == NS_HOST) NS_CK(cudaStreamSynchronize(st));
        return NS_OK;
    }

    int padded_size() const override { return M; }
    int transform_grid() const override { return N; }

    // autotune probe: milliseconds of one pass a1..a6 over whatever the workspaces hold (the work is data independent)
    int time_transform(int reps, double* ms) override {
        cudaEvent_t a, b;
        NS_CK(cudaEventCreate(&a));
        NS_CK(cudaEventCreate(&b));
        NS_CK(cudaMemsetAsync(U, 0, nS * sizeof(cx<T>), st));
        int rc = transform(U, false);
        if (rc == NS_OK) {
            cudaEventRecord(a, st);
            for (int i = 0; i < reps && rc == NS_OK; ++i) rc = transform(U, false);
            cudaEventRecord(b, st);
            cudaError_t e = cudaStreamSynchronize(st);
            float t = 0;
            if (rc == NS_OK && e == cudaSuccess && cudaEventElapsedTime(&t, a, b) == cudaSuccess) *ms = t / reps;
            else if (rc == NS_OK) rc = cuda_fail(e, "time_transform");
        }
        cudaEventDestroy(a);
        cudaEventDestroy(b);
        return rc;
    }

    int profile(int enable) override {
        NS_CK(cudaStreamSynchronize(st));
        prof.reset();
        prof.on = enable != 0;
        if (prof.on) prof.reserve(512);
        return NS_OK;
    }
    int profile_read(double* ms, long long* cnt) override {
        if (!ms || !cnt) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        NS_CK(cudaStreamSynchronize(st));
        prof.collect();
        for (int i = 0; i < PassProfiler::NPASS; ++i) { ms[i] = prof.ms[i]; cnt[i] = prof.cnt[i]; }
        return NS_OK;
    }

    double time(int sample) override {
        if (sample < 0 || sample >= batch) return std::numeric_limits<double>::quiet_NaN();
        double t = 0.0;
        if (cudaMemcpyAsync(&t, t_dev + sample, sizeof(double), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
            cudaStreamSynchronize(st) != cudaSuccess)
            return std::numeric_limits<double>::quiet_NaN();
        return t;
    }
};

template <typename T>
int create_typed(ns_solver** out, int Nu, int N, int batch, const ns_params& p, cudaStream_t st) {
    Solver<T>* s = new Solver<T>(Nu, N, batch, p, st);
    int rc = s->init();
    if (rc != NS_OK) {
        g_create_error = s->err;
        delete s;
        return rc;
    }
    *out = s;
    return NS_OK;
}

// ---- transform-grid selection ("we round the padded data's size up to the next value of the form 2^a 3^b 5^c 7^d
// ... On any new system, we therefore once run a benchmark of only the Fourier transform storing its results and extracting the
// optimal padding size from that generated data.  If no suitable size is found in the benchmark results, we choose the next
// larger N with prime factors at most 7 instead").  Here the padded grid is 3/2 of the TRANSFORM grid Nt >= N, Nt/2 one of the
// supported lengths; the state lives on the Nt grid with zeros outside K_N, which gives the RHS of the user's N exactly
// (independence of the padding, oracle pin P7).
bool transform_grid_ok(int Nt, ns_dtype dtype) {
    const int tile = dtype == NS_F32 ? 16 : 8;
    return Nt >= 16 && Nt <= 640 && Nt % 2 == 0 && fft_supported(Nt / 2) && (Nt / 2) % tile == 0;
}
int next_transform_grid(int N, ns_dtype dtype) {
    for (int Nt = N + (N & 1); Nt <= 640; Nt += 2)
        if (transform_grid_ok(Nt, dtype)) return Nt;
    return 0;
}
struct TuneKey {
    int device, N, dtype;
    bool operator<(const TuneKey& o) const { return device != o.device ? device < o.device : (N != o.N ? N < o.N : dtype < o.dtype); }
};
std::mutex g_tune_mutex;
std::map<TuneKey, int> g_tune_table;   // (device, N, dtype) -> transform grid chosen by ns_autotune

}  // namespace

extern "C" {

static int resolve_params(const ns_params* p, ns_params* prm) {
    std::memset(prm, 0, sizeof *prm);
    prm->s = 1.0;
    prm->m_cut = -1.0;
    prm->q_exp = -1.0;
    if (p) *prm = *p;
    if (!(prm->s >= 1.0) || prm->nu < 0.0 || prm->eps < 0.0 || !(prm->nu == prm->nu) || !(prm->eps == prm->eps)) {
        g_create_error = "params: need s >= 1, nu >= 0, eps >= 0";
        return NS_ERR_INVALID_ARG;
    }
    return NS_OK;
}
static int create_on_grid(ns_solver** out, int N, int Nt, int batch, const ns_params* p, ns_dtype dtype, void* cuda_stream) {
    ns_params prm;
    int rcp = resolve_params(p, &prm);
    if (rcp != NS_OK) return rcp;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return dtype == NS_F64 ? create_typed<double>(out, N, Nt, batch, prm, st) : create_typed<float>(out, N, Nt, batch, prm, st);
}
static int check_device() {
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        g_create_error = std::string("no usable CUDA device (no CPU fallback): ") + (e != cudaSuccess ? cudaGetErrorString(e) : "0 devices");
        return NS_ERR_CUDA;
    }
    return NS_OK;
}
static int check_sizes(int N, int batch, ns_dtype dtype) {
    if (dtype != NS_F64 && dtype != NS_F32) { g_create_error = "unknown dtype"; return NS_ERR_INVALID_ARG; }
    // any even N; the transforms run on the next grid Nt >= N with Nt = p 2^a, p in {1, 3, 5, 7, 15}, Nt/2 a multiple of the
    // column tile (128 bytes = 8 fp64 / 16 fp32 complex values)
    if (N < 16 || N > 640 || (N % 2) != 0 || next_transform_grid(N, dtype) == 0) {
        g_create_error = "N must be even with 16 <= N <= 640";
        return NS_ERR_INVALID_ARG;
    }
    if (batch < 1) { g_create_error = "batch must be >= 1"; return NS_ERR_INVALID_ARG; }
    return NS_OK;
}

int ns_create(ns_solver** out, int N, int batch, const ns_params* p, ns_dtype dtype, void* cuda_stream) {
    g_create_error.clear();
    if (!out) { g_create_error = "out is NULL"; return NS_ERR_INVALID_ARG; }
    *out = nullptr;
    int rc = check_sizes(N, batch, dtype);
    if (rc != NS_OK) return rc;
    ns_params chk;
    if ((rc = resolve_params(p, &chk)) != NS_OK) return rc;
    if ((rc = check_device()) != NS_OK) return rc;
    int Nt = next_transform_grid(N, dtype), dev = 0;
    cudaGetDevice(&dev);
    {
        std::lock_guard<std::mutex> lock(g_tune_mutex);
        auto it = g_tune_table.find(TuneKey{dev, N, (int)dtype});
        if (it != g_tune_table.end()) Nt = it->second;
    }
    return create_on_grid(out, N, Nt, batch, p, dtype, cuda_stream);
}

int ns_autotune(int N, ns_dtype dtype, int ncand, int* grids_out, double* ms_out, int* best_out) {
    g_create_error.clear();
    int rc = check_sizes(N, 1, dtype);
    if (rc != NS_OK) return rc;
    if (ncand < 1 || ncand > 16) { g_create_error = "ncand must be in [1, 16]"; return NS_ERR_INVALID_ARG; }
    if ((rc = check_device()) != NS_OK) return rc;
    int best = 0, found = 0;
    double best_ms = 0.0;
    for (int Nt = next_transform_grid(N, dtype); Nt != 0 && found < ncand; Nt = next_transform_grid(Nt + 2, dtype)) {
        ns_solver* h = nullptr;
        rc = create_on_grid(&h, N, Nt, 1, nullptr, dtype, nullptr);
        double ms = 0.0;
        if (rc == NS_OK) rc = h->time_transform(3, &ms);
        if (rc != NS_OK && h) g_create_error = h->err;
        delete h;
        if (rc == NS_ERR_OOM && found > 0) break;      // larger grids do not fit: keep what was measured
        if (rc != NS_OK) return rc;
        if (grids_out) grids_out[found] = Nt;
        if (ms_out) ms_out[found] = ms;
        if (found == 0 || ms < best_ms) { best = Nt; best_ms = ms; }
        ++found;
    }
    for (int i = found; i < ncand; ++i) {
        if (grids_out) grids_out[i] = 0;
        if (ms_out) ms_out[i] = 0.0;
    }
    int dev = 0;
    cudaGetDevice(&dev);
    {
        std::lock_guard<std::mutex> lock(g_tune_mutex);
        g_tune_table[TuneKey{dev, N, (int)dtype}] = best;
    }
    if (best_out) *best_out = best;
    return NS_OK;
}

int ns_destroy(ns_solver* h) {
    if (!h) return NS_ERR_INVALID_ARG;
    delete h;
    return NS_OK;
}

#define NS_H(h) if (!(h)) return NS_ERR_INVALID_ARG; (h)->err.clear()

int ns_set_initial(ns_solver* h, const void* u, ns_memspace ms) { NS_H(h); return h->set_initial(u, ms); }
int ns_set_spectral(ns_solver* h, const void* u, ns_memspace ms) { NS_H(h); return h->set_spectral(u, ms); }
int ns_get_spectral(ns_solver* h, void* u, ns_memspace ms) { NS_H(h); return h->get_spectral(u, ms); }
int ns_rhs(ns_solver* h, void* out, ns_memspace ms) { NS_H(h); return h->rhs(out, ms); }
int ns_step(ns_solver* h, double dt) { NS_H(h); return h->step_uniform(dt); }
int ns_step_cfl(ns_solver* h, double cfl, double t_end, double* dt_out) { NS_H(h); return h->step_cfl(cfl, t_end, dt_out); }
int ns_step_dts(ns_solver* h, const double* dt) { NS_H(h); return h->step_dts(dt); }
int ns_advance(ns_solver* h, double cfl, double t_end, int max_steps, int* steps_done) { NS_H(h); return h->advance(cfl, t_end, max_steps, steps_done); }
int ns_max_velocity(ns_solver* h, double* out) { NS_H(h); return h->max_velocity(out); }
int ns_get_fields(ns_solver* h, void* out, ns_memspace ms) { NS_H(h); return h->get_fields(out, ms); }
int ns_energy_spectrum(ns_solver* h, double* E, int nbins) { NS_H(h); return h->energy_spectrum(E, nbins, false); }
int ns_enstrophy_spectrum(ns_solver* h, double* Z, int nbins) { NS_H(h); return h->energy_spectrum(Z, nbins, true); }
int ns_structure_function(ns_solver* h, double* S, int nl) { NS_H(h); return h->structure_function(S, nl); }
int ns_ensemble_moments(ns_solver* h, void* mean, void* var, ns_memspace ms) { NS_H(h); return h->ensemble_moments(mean, var, ms); }
int ns_structure_function_p(ns_solver* h, double p, double* S, int nl) { NS_H(h); return h->structure_function_p(p, S, nl); }
double ns_time(const ns_solver* h, int sample) {
    if (!h) return std::numeric_limits<double>::quiet_NaN();
    return const_cast<ns_solver*>(h)->time(sample);
}
int ns_profile(ns_solver* h, int enable) { NS_H(h); return h->profile(enable); }
int ns_profile_read(ns_solver* h, double* ms, long long* cnt) { NS_H(h); return h->profile_read(ms, cnt); }
int ns_transform_grid(const ns_solver* h) { return h ? h->transform_grid() : 0; }
int ns_padded_size(const ns_solver* h) { return h ? h->padded_size() : 0; }
long long ns_kernel_launches(const ns_solver* h) { return h ? h->launches : 0; }
long long ns_device_bytes(const ns_solver* h) { return h ? h->device_bytes() : 0; }
const char* ns_last_error(const ns_solver* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

}  // extern "C"
