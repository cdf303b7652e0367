// ns2d_solver.cu -- host side of the TWO-DIMENSIONAL solver (include/ns2d.h): handle, workspace arena and
// the launch sequences.  One RHS = 4 launches: b1 pad + inverse transform along x (the strided-axis kernels of kernels_col.cuh),
// b2 the fused y kernel (kernels_y2d.cuh: inverse, trace-free flux, forward), b3 forward along x + truncate, b4 the spectral
// kernel (kernels_misc2d.cuh).  Launches only; no CPU fallback.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <limits>
#include <string>
#include <vector>

#include "../../include/ns2d.h"
#include "kernels_misc2d.cuh"
#include "ns_internal.h"
#include "twiddles_host.h"

using namespace ns;

struct ns2d_solver {
    std::string err;
    long long launches = 0;
    virtual ~ns2d_solver() {}
    virtual int set_initial(const void* u, ns_memspace ms) = 0;
    virtual int set_spectral(const void* u, ns_memspace ms) = 0;
    virtual int get_spectral(void* u, ns_memspace ms) = 0;
    virtual int rhs(void* out, ns_memspace ms) = 0;
    virtual int step(int mode, double dt, const double* dts, double cfl, double t_end, double* dt_out) = 0;
    virtual int advance(double cfl, double t_end, int max_steps, int* steps_done) = 0;
    virtual int max_velocity(double* out) = 0;
    virtual int get_fields(void* out, ns_memspace ms) = 0;
    virtual int spectrum(double* E, int nbins, bool enstrophy) = 0;
    virtual double time(int sample) = 0;
    virtual long long device_bytes() const = 0;
    virtual int transform_grid() const = 0;
    virtual int profile(int enable) = 0;
    virtual int profile_read(double* ms, long long* cnt) = 0;
};

static thread_local std::string g_create_error2d;

namespace {

double dissipation_rate2d(const ns_params& p, int N, double k2) {
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

enum { DT_UNIFORM = 0, DT_ARRAY = 1, DT_CFL = 2 };

template <typename T>
class Solver2D final : public ns2d_solver {
public:
    int N, L, M, H, batch;   // N = the transform grid (128, 256 or 512), M = 3N/2 its padded grid
    int Nu;                  // the user's grid (public arrays, truncation set, dx, eps_N, m_N); Nu <= N
    cx<T>* gNu = nullptr;    // exp(2 pi i j / Nu), j < Nu
    int device = 0, num_sms = 0;
    ns_params prm;
    cudaStream_t st;
    bool has_state = false;
    unsigned char* arena = nullptr;
    size_t arena_bytes = 0;
    cx<T>*U = nullptr, *V = nullptr, *X = nullptr, *Y = nullptr, *Z = nullptr;
    cx<T>* twbase = nullptr;
    T* dtab = nullptr;
    double *dt_dev = nullptr, *t_dev = nullptr, *scal_dev = nullptr, *red_dev = nullptr;
    unsigned long long* umax2 = nullptr;
    int* bad_dev = nullptr;
    // per-pass profiler: 0 x inverse, 1 fused y, 2 x forward, 3 spectral
    bool prof_on = false;
    std::vector<cudaEvent_t> ev;
    std::vector<int> tag;
    size_t used = 0;
    double pms[4] = {0, 0, 0, 0};
    long long pcnt[4] = {0, 0, 0, 0};

    Solver2D(int Nu_, int N_, int batch_, const ns_params& p, cudaStream_t s)
        : N(N_), L(N_ / 2), M(3 * N_ / 2), H(N_ / 2), batch(batch_), Nu(Nu_), prm(p), st(s) {}
    ~Solver2D() override {
        for (cudaEvent_t e : ev) cudaEventDestroy(e);
        if (arena) cudaFree(arena);
    }
    int fail(int code, const std::string& msg) { err = msg; return code; }
    int cuda_fail(cudaError_t e, const char* where) { err = std::string(where) + ": " + cudaGetErrorString(e); return NS_ERR_CUDA; }
#define NS_CK(call)                                           \
    do {                                                      \
        cudaError_t e__ = (call);                             \
        if (e__ != cudaSuccess) return cuda_fail(e__, #call); \
    } while (0)
#define NS_LAUNCHED(name)                                    \
    do {                                                     \
        ++launches;                                          \
        cudaError_t e__ = cudaGetLastError();                \
        if (e__ != cudaSuccess) return cuda_fail(e__, name); \
    } while (0)

    void tick(int pass) {
        if (!prof_on || used >= ev.size()) return;
        tag[used] = pass;
        cudaEventRecord(ev[used], st);
        ++used;
    }
    Twiddles<T> tw() const { return make_twiddles<T>(twbase, L); }
    static unsigned blocks_for(long total, int threads) { return (unsigned)((total + threads - 1) / threads); }

    int init() {
        NS_CK(cudaGetDevice(&device));
        NS_CK(cudaDeviceGetAttribute(&num_sms, cudaDevAttrMultiProcessorCount, device));
        const size_t b = (size_t)batch;
        const size_t nS = b * 2 * N * H;
        size_t nX = b * 2 * (size_t)M * H;          // b1 out; also the full complex planes of the unpadded transforms
        if (nX < b * 2 * (size_t)N * N) nX = b * 2 * (size_t)N * N;
        size_t nY = b * 2 * (size_t)N * (H + 1);    // b3 out (T_hat, 2 N H); public-layout / physical staging
        if (nY < b * (size_t)N * N) nY = b * (size_t)N * N;
        const size_t nZ = b * 2 * (size_t)M * H;    // b2 out
        const size_t ndt = (size_t)2 * L * L + 1;
        auto al = [](size_t x) { return (x + 255) & ~(size_t)255; };
        size_t off = 0;
        auto take = [&](size_t bytes) { size_t o = off; off += al(bytes); return o; };
        const size_t oU = take(nS * sizeof(cx<T>)), oV = take(nS * sizeof(cx<T>));
        const size_t oX = take(nX * sizeof(cx<T>)), oY = take(nY * sizeof(cx<T>)), oZ = take(nZ * sizeof(cx<T>));
        const size_t otw = take(twiddle_table_len(L) * sizeof(cx<T>));
        const size_t ogu = take((size_t)Nu * sizeof(cx<T>));
        const size_t oD = take(ndt * sizeof(T));
        const size_t odt = take(b * sizeof(double)), ot = take(b * sizeof(double)), osc = take(b * sizeof(double));
        const size_t oum = take(b * sizeof(unsigned long long)), obad = take(b * sizeof(int));
        const size_t ored = take(b * 4096 * sizeof(double));
        arena_bytes = off;
        cudaError_t e = cudaMalloc(&arena, arena_bytes);
        if (e == cudaErrorMemoryAllocation) {
            cudaGetLastError();
            char buf[128];
            snprintf(buf, sizeof buf, "device allocation of %.2f GB failed", (double)arena_bytes / 1e9);
            return fail(NS_ERR_OOM, buf);
        }
        if (e != cudaSuccess) return cuda_fail(e, "cudaMalloc");
        U = (cx<T>*)(arena + oU); V = (cx<T>*)(arena + oV); X = (cx<T>*)(arena + oX); Y = (cx<T>*)(arena + oY); Z = (cx<T>*)(arena + oZ);
        twbase = (cx<T>*)(arena + otw);
        gNu = (cx<T>*)(arena + ogu);
        dtab = (T*)(arena + oD);
        dt_dev = (double*)(arena + odt); t_dev = (double*)(arena + ot); scal_dev = (double*)(arena + osc);
        umax2 = (unsigned long long*)(arena + oum);
        bad_dev = (int*)(arena + obad);
        red_dev = (double*)(arena + ored);
        const std::vector<cx<T>> htw = build_twiddle_block<T>(L);
        std::vector<T> hd(ndt);
        for (size_t k2 = 0; k2 < ndt; ++k2) hd[k2] = (T)dissipation_rate2d(prm, Nu, (double)k2);   // eps_N, m_N of the USER's N
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
    int transform_grid() const override { return N; }

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

    // Uin (internal layout) -> Y = T_hat [b][2][N][H] (unnormalised transforms of T11, T12)
    int transform(const cx<T>* Uin, bool want_umax, int upto = 3) {
        const long MH = (long)M * H, NH = (long)N * H;
        cudaError_t e;
        tick(0);
        e = launch_col_inv<T>(st, num_sms, L, Uin, X, H, (long)batch * 2, H, H, NH, MH, tw());
        if (e != cudaSuccess) return cuda_fail(e, "b1 col_inv x");
        ++launches;
        tick(1);
        e = launch_y2d<T>(st, num_sms, L, X, Z, M, batch, want_umax ? umax2 : nullptr, tw());
        if (e != cudaSuccess) return cuda_fail(e, "b2 y2d");
        ++launches;
        if (upto <= 2) { tick(-1); return NS_OK; }
        tick(2);
        e = launch_col_fwd<T>(st, num_sms, L, Z, Y, H, (long)batch * 2, H, H, MH, NH, (T)1, tw());
        if (e != cudaSuccess) return cuda_fail(e, "b3 col_fwd x");
        ++launches;
        tick(-1);
        return NS_OK;
    }
    int spectral(const cx<T>* Us, const cx<T>* Un, cx<T>* out, double alpha, double beta, double gamma, int mode) {
        const long total = (long)batch * N * H;
        const T scale = (T)(1.0 / ((double)M * M * z_fused_output_scale(L)));
        tick(3);
        spectral2d_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(Y, Us, Un, out, N, Nu / 2, total, dtab, scale, (T)alpha, (T)beta, (T)gamma,
                                                                      dt_dev, mode);
        NS_LAUNCHED("b4 spectral2d_kernel");
        tick(-1);
        return NS_OK;
    }

    int rk3(int mode, double dt, const double* dts_host, double cfl, double t_end) {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        int rc;
        const unsigned gb = blocks_for(batch, 128);
        NS_CK(cudaMemsetAsync(umax2, 0, (size_t)batch * sizeof(unsigned long long), st));
        if ((rc = transform(U, true)) != NS_OK) return rc;
        if (mode == DT_UNIFORM) {
            set_dt_uniform_kernel<<<gb, 128, 0, st>>>(dt_dev, t_dev, dt, umax2, bad_dev, batch);
            NS_LAUNCHED("set_dt_uniform");
        } else if (mode == DT_ARRAY) {
            NS_CK(cudaMemcpyAsync(scal_dev, dts_host, (size_t)batch * sizeof(double), cudaMemcpyHostToDevice, st));
            set_dt_array_kernel<<<gb, 128, 0, st>>>(dt_dev, t_dev, scal_dev, umax2, bad_dev, batch);
            NS_LAUNCHED("set_dt_array");
        } else {
            cfl_finalize_kernel<<<gb, 128, 0, st>>>(dt_dev, t_dev, umax2, bad_dev, cfl, 2.0 * 3.14159265358979323846 / Nu, t_end, batch);
            NS_LAUNCHED("cfl_finalize");
        }
        if ((rc = spectral(U, nullptr, V, 0.0, 1.0, 1.0, 1)) != NS_OK) return rc;                       // u1 = u + dt R(u)
        if ((rc = transform(V, false)) != NS_OK) return rc;
        if ((rc = spectral(V, U, V, 0.75, 0.25, 0.25, 1)) != NS_OK) return rc;                          // u2 = 3/4 u + 1/4 u1 + 1/4 dt R(u1)
        if ((rc = transform(V, false)) != NS_OK) return rc;
        return spectral(V, U, U, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, 1);                                    // u+ = 1/3 u + 2/3 u2 + 2/3 dt R(u2)
    }

    int step(int mode, double dt, const double* dts, double cfl, double t_end, double* dt_out) override {
        if (mode == DT_UNIFORM && (!(dt == dt) || std::isinf(dt))) return fail(NS_ERR_INVALID_ARG, "dt must be finite");
        if (mode == DT_ARRAY && !dts) return fail(NS_ERR_INVALID_ARG, "dt array is NULL");
        if (mode == DT_CFL && !(cfl > 0.0)) return fail(NS_ERR_INVALID_ARG, "cfl must be positive");
        int rc = rk3(mode, dt, dts, cfl, t_end);
        if (rc != NS_OK) return rc;
        if (mode == DT_ARRAY) return check_finite();
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
            int rcf = check_finite();
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
        int rc = transform(U, true, 2);
        if (rc != NS_OK) return rc;
        umax_read_kernel<<<blocks_for(batch, 128), 128, 0, st>>>(scal_dev, umax2, bad_dev, batch);
        NS_LAUNCHED("umax_read");
        NS_CK(cudaMemcpyAsync(out, scal_dev, (size_t)batch * sizeof(double), cudaMemcpyDeviceToHost, st));
        return check_finite();
    }

    int export_spectral(const cx<T>* src, void* out, ns_memspace ms) {
        const long total_pub = (long)batch * 2 * Nu * (Nu / 2 + 1);
        cx<T>* dst = ms == NS_DEVICE ? (cx<T>*)out : Y;
        to_public2d_kernel<T><<<blocks_for(total_pub, 256), 256, 0, st>>>(src, dst, N, Nu, total_pub);
        NS_LAUNCHED("to_public2d");
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(out, Y, (size_t)total_pub * sizeof(cx<T>), cudaMemcpyDeviceToHost, st));
            NS_CK(cudaStreamSynchronize(st));
        }
        return NS_OK;
    }
    int rhs(void* out, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        int rc = transform(U, false);
        if (rc != NS_OK) return rc;
        if ((rc = spectral(U, nullptr, X, 0, 0, 0, 0)) != NS_OK) return rc;
        return export_spectral(X, out, ms);
    }
    int get_spectral(void* out, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        return export_spectral(U, out, ms);
    }
    int set_spectral(const void* in, ns_memspace ms) override {
        if (!in) return fail(NS_ERR_INVALID_ARG, "input pointer is NULL");
        const long total_pub = (long)batch * 2 * Nu * (Nu / 2 + 1);
        const cx<T>* src = (const cx<T>*)in;
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(Y, in, (size_t)total_pub * sizeof(cx<T>), cudaMemcpyHostToDevice, st));
            src = Y;
        }
        const long total = (long)batch * 2 * N * H;
        to_internal2d_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(src, U, N, Nu, total);
        NS_LAUNCHED("to_internal2d");
        NS_CK(cudaMemsetAsync(bad_dev, 0, (size_t)batch * sizeof(int), st));
        if (ms == NS_HOST) NS_CK(cudaStreamSynchronize(st));
        has_state = true;
        return NS_OK;
    }

    // unpadded 2-D transform on the USER's grid (planes of Nu^2 complex), in place: mixed radix when Nu = p 2^a with p in
    // {1, 3, 5, 7, 15} and Nu a multiple of 8, else the plain DFT
    int generic_fft2(cx<T>* W, long planes, int sign) {
        int odd = Nu, log2m = 0;
        while (odd % 2 == 0) { odd /= 2; ++log2m; }
        const bool fast = (odd == 1 || odd == 3 || odd == 5 || odd == 7 || odd == 15) && Nu % 8 == 0;
        if (fast) {
            const long tiles = planes * (long)Nu / 8;
            const size_t smem = (size_t)Nu * 9 * sizeof(cx<T>);
            if (smem > 48 * 1024)
                NS_CK(cudaFuncSetAttribute(generic_fft_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            for (int axis = 1; axis < 3; ++axis) {
                generic_fft_kernel<T><<<(unsigned)tiles, 256, smem, st>>>(W, Nu, log2m, odd, axis, sign, tiles, gNu, 2);
                NS_LAUNCHED("generic_fft 2d");
            }
        } else {
            const long tiles = planes * (((long)Nu + 7) / 8);
            const size_t smem = (size_t)2 * Nu * 9 * sizeof(cx<T>);
            if (smem > 48 * 1024)
                NS_CK(cudaFuncSetAttribute(dft_lines_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
            for (int axis = 1; axis < 3; ++axis) {
                dft_lines_kernel<T><<<(unsigned)tiles, 256, smem, st>>>(W, Nu, axis, sign, tiles, gNu, 2);
                NS_LAUNCHED("dft_lines 2d");
            }
        }
        return NS_OK;
    }
    int set_initial(const void* in, ns_memspace ms) override {
        if (!in) return fail(NS_ERR_INVALID_ARG, "input pointer is NULL");
        const long planes = (long)batch * 2;
        const long total = planes * Nu * Nu;
        const T* src = (const T*)in;
        if (ms == NS_HOST) {
            NS_CK(cudaMemcpyAsync(Y, in, (size_t)total * sizeof(T), cudaMemcpyHostToDevice, st));
            src = reinterpret_cast<const T*>(Y);
        }
        real_to_complex_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(src, X, total);
        NS_LAUNCHED("real_to_complex");
        int rc = generic_fft2(X, planes, -1);
        if (rc != NS_OK) return rc;
        const long tot = (long)batch * N * H;
        init_project2d_kernel<T><<<blocks_for(tot, 256), 256, 0, st>>>(X, U, N, Nu, tot, (T)(1.0 / ((double)Nu * Nu)));
        NS_LAUNCHED("init_project2d");
        NS_CK(cudaMemsetAsync(t_dev, 0, (size_t)batch * sizeof(double), st));
        NS_CK(cudaMemsetAsync(bad_dev, 0, (size_t)batch * sizeof(int), st));
        if (ms == NS_HOST) NS_CK(cudaStreamSynchronize(st));
        has_state = true;
        return NS_OK;
    }
    int get_fields(void* out, ns_memspace ms) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!out) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        const long planes = (long)batch * 2;
        const long total = planes * Nu * Nu;
        expand_hermitian2d_kernel<T><<<blocks_for(total, 256), 256, 0, st>>>(U, X, N, Nu, total);
        NS_LAUNCHED("expand_hermitian2d");
        int rc = generic_fft2(X, planes, +1);
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
    int spectrum(double* E, int nbins, bool enstrophy) override {
        if (!has_state) return fail(NS_ERR_STATE, "no initial state set");
        if (!E || nbins < 1 || nbins > 4096) return fail(NS_ERR_INVALID_ARG, "E is NULL or nbins not in [1, 4096]");
        NS_CK(cudaMemsetAsync(red_dev, 0, (size_t)batch * nbins * sizeof(double), st));
        const long plane = (long)N * H;
        unsigned chunks = blocks_for(plane, 256 * 16);
        if (chunks > 64) chunks = 64;
        const unsigned by = (unsigned)batch;   // gridDim.y <= 65535
        if (by > 65535) return fail(NS_ERR_INVALID_ARG, "batch too large for the spectrum kernel");
        if (enstrophy)
            spectrum2d_kernel<T, true><<<dim3(chunks, by), 256, (size_t)nbins * sizeof(double), st>>>(U, red_dev, N, nbins);
        else
            spectrum2d_kernel<T, false><<<dim3(chunks, by), 256, (size_t)nbins * sizeof(double), st>>>(U, red_dev, N, nbins);
        NS_LAUNCHED("spectrum2d");
        NS_CK(cudaMemcpyAsync(E, red_dev, (size_t)batch * nbins * sizeof(double), cudaMemcpyDeviceToHost, st));
        NS_CK(cudaStreamSynchronize(st));
        return NS_OK;
    }

    int profile(int enable) override {
        NS_CK(cudaStreamSynchronize(st));
        used = 0;
        for (int i = 0; i < 4; ++i) { pms[i] = 0; pcnt[i] = 0; }
        prof_on = enable != 0;
        while (prof_on && ev.size() < 512) {
            cudaEvent_t e;
            NS_CK(cudaEventCreate(&e));
            ev.push_back(e);
            tag.push_back(-1);
        }
        return NS_OK;
    }
    int profile_read(double* ms, long long* cnt) override {
        if (!ms || !cnt) return fail(NS_ERR_INVALID_ARG, "output pointer is NULL");
        NS_CK(cudaStreamSynchronize(st));
        for (size_t i = 0; i + 1 < used; ++i) {
            if (tag[i] < 0) continue;
            float t = 0;
            if (cudaEventElapsedTime(&t, ev[i], ev[i + 1]) == cudaSuccess) { pms[tag[i]] += t; pcnt[tag[i]] += 1; }
        }
        used = 0;
        for (int i = 0; i < 4; ++i) { ms[i] = pms[i]; cnt[i] = pcnt[i]; }
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
int create_typed2d(ns2d_solver** out, int Nu, int N, int batch, const ns_params& p, cudaStream_t st) {
    Solver2D<T>* s = new Solver2D<T>(Nu, N, batch, p, st);
    int rc = s->init();
    if (rc != NS_OK) {
        g_create_error2d = s->err;
        delete s;
        return rc;
    }
    *out = s;
    return NS_OK;
}

}  // namespace

extern "C" {

int ns2d_create(ns2d_solver** out, int N, int batch, const ns_params* p, ns_dtype dtype, void* cuda_stream) {
    g_create_error2d.clear();
    if (!out) { g_create_error2d = "out is NULL"; return NS_ERR_INVALID_ARG; }
    *out = nullptr;
    // any even N up to 512; the transforms run on the next transform grid Nt in {128, 256, 512} (the padded size is
    // rounded up to one the transforms are fast for), the state truncated to the user's N -- as ns.h
    if (N < 16 || N > 512 || (N % 2) != 0) { g_create_error2d = "N must be even with 16 <= N <= 512"; return NS_ERR_INVALID_ARG; }
    const int Nt = N <= 128 ? 128 : (N <= 256 ? 256 : 512);
    if (batch < 1) { g_create_error2d = "batch must be >= 1"; return NS_ERR_INVALID_ARG; }
    if ((long)batch * (3 * Nt / 2) >= (1L << 31)) { g_create_error2d = "batch too large"; return NS_ERR_INVALID_ARG; }
    if (dtype != NS_F64 && dtype != NS_F32) { g_create_error2d = "unknown dtype"; return NS_ERR_INVALID_ARG; }
    ns_params prm;
    std::memset(&prm, 0, sizeof prm);
    prm.s = 1.0;
    prm.m_cut = -1.0;
    prm.q_exp = -1.0;
    if (p) prm = *p;
    if (!(prm.s >= 1.0) || prm.nu < 0.0 || prm.eps < 0.0 || !(prm.nu == prm.nu) || !(prm.eps == prm.eps)) {
        g_create_error2d = "params: need s >= 1, nu >= 0, eps >= 0";
        return NS_ERR_INVALID_ARG;
    }
    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        g_create_error2d = std::string("no usable CUDA device (no CPU fallback): ") + (e != cudaSuccess ? cudaGetErrorString(e) : "0 devices");
        return NS_ERR_CUDA;
    }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    return dtype == NS_F64 ? create_typed2d<double>(out, N, Nt, batch, prm, st) : create_typed2d<float>(out, N, Nt, batch, prm, st);
}
int ns2d_destroy(ns2d_solver* h) {
    if (!h) return NS_ERR_INVALID_ARG;
    delete h;
    return NS_OK;
}
#define NS2_H(h) if (!(h)) return NS_ERR_INVALID_ARG; (h)->err.clear()
int ns2d_set_initial(ns2d_solver* h, const void* u, ns_memspace ms) { NS2_H(h); return h->set_initial(u, ms); }
int ns2d_set_spectral(ns2d_solver* h, const void* u, ns_memspace ms) { NS2_H(h); return h->set_spectral(u, ms); }
int ns2d_get_spectral(ns2d_solver* h, void* u, ns_memspace ms) { NS2_H(h); return h->get_spectral(u, ms); }
int ns2d_rhs(ns2d_solver* h, void* out, ns_memspace ms) { NS2_H(h); return h->rhs(out, ms); }
int ns2d_step(ns2d_solver* h, double dt) { NS2_H(h); return h->step(DT_UNIFORM, dt, nullptr, 0, 0, nullptr); }
int ns2d_step_cfl(ns2d_solver* h, double cfl, double t_end, double* dt_out) { NS2_H(h); return h->step(DT_CFL, 0, nullptr, cfl, t_end, dt_out); }
int ns2d_step_dts(ns2d_solver* h, const double* dt) { NS2_H(h); return h->step(DT_ARRAY, 0, dt, 0, 0, nullptr); }
int ns2d_advance(ns2d_solver* h, double cfl, double t_end, int max_steps, int* steps_done) { NS2_H(h); return h->advance(cfl, t_end, max_steps, steps_done); }
int ns2d_max_velocity(ns2d_solver* h, double* out) { NS2_H(h); return h->max_velocity(out); }
int ns2d_get_fields(ns2d_solver* h, void* out, ns_memspace ms) { NS2_H(h); return h->get_fields(out, ms); }
int ns2d_energy_spectrum(ns2d_solver* h, double* E, int nbins) { NS2_H(h); return h->spectrum(E, nbins, false); }
int ns2d_enstrophy_spectrum(ns2d_solver* h, double* Z, int nbins) { NS2_H(h); return h->spectrum(Z, nbins, true); }
double ns2d_time(const ns2d_solver* h, int sample) {
    if (!h) return std::numeric_limits<double>::quiet_NaN();
    return const_cast<ns2d_solver*>(h)->time(sample);
}
int ns2d_profile(ns2d_solver* h, int enable) { NS2_H(h); return h->profile(enable); }
int ns2d_profile_read(ns2d_solver* h, double* ms, long long* cnt) { NS2_H(h); return h->profile_read(ms, cnt); }
int ns2d_transform_grid(const ns2d_solver* h) { return h ? h->transform_grid() : 0; }
long long ns2d_kernel_launches(const ns2d_solver* h) { return h ? h->launches : 0; }
long long ns2d_device_bytes(const ns2d_solver* h) { return h ? h->device_bytes() : 0; }
const char* ns2d_last_error(const ns2d_solver* h) { return h ? h->err.c_str() : g_create_error2d.c_str(); }

}  // extern "C"
