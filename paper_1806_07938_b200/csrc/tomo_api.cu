// tomo_api.cu -- C ABI of libtomo_b200 (include/tomo.h): plan life cycle, kernel-spectra upload, and the
// launch sequences of rows A1-A8.  No CPU fallback: every compute entry point needs the CUDA device.
#include <cmath>
#include <complex>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <type_traits>
#include <vector>

#include "tomo.h"
#include "tomo_kernels.cuh"
#include "tomo_kernels_cos.cuh"
#include "tomo_kernels_minres.cuh"
#include "tomo_plan.hpp"

namespace tomo {
static thread_local std::string g_err;
void set_error(const std::string &s) { g_err = s; }

#define CK(call)                                                                                        \
    do {                                                                                                \
        cudaError_t e_ = (call);                                                                        \
        if (e_ != cudaSuccess) {                                                                        \
            set_error(std::string(#call) + ": " + cudaGetErrorString(e_));                              \
            return TOMO_ECUDA;                                                                          \
        }                                                                                               \
    } while (0)

static void plan_fft(int P, FftDesc &d) {
    d.P = P; d.nrad = 0;
    int r = P;
    while (r % 5 == 0) { d.rad[d.nrad++] = 5; r /= 5; }
    while (r % 3 == 0) { d.rad[d.nrad++] = 3; r /= 3; }
    while (r % 8 == 0) { d.rad[d.nrad++] = 8; r /= 8; }
    while (r % 4 == 0) { d.rad[d.nrad++] = 4; r /= 4; }
    while (r % 2 == 0) { d.rad[d.nrad++] = 2; r /= 2; }
}

template <typename V> static int dev_alloc(tomo_plan *pl, V **ptr, size_t count) {
    void *p = nullptr;
    const size_t bytes = std::max<size_t>(count, 1) * sizeof(V);
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { set_error(std::string("cudaMalloc: ") + cudaGetErrorString(e)); return TOMO_ENOMEM; }
    pl->allocs.push_back(p);
    pl->bytes += bytes;
    *ptr = reinterpret_cast<V *>(p);
    return TOMO_OK;
}
static int dev_alloc_bytes(tomo_plan *pl, void **ptr, size_t bytes) {
    unsigned char *p = nullptr;
    int rc = dev_alloc<unsigned char>(pl, &p, bytes);
    *ptr = p;
    return rc;
}
template <typename V> static int upload(tomo_plan *pl, V **ptr, const std::vector<V> &h) {
    int rc = dev_alloc<V>(pl, ptr, h.size());
    if (rc) return rc;
    if (!h.empty()) CK(cudaMemcpy(*ptr, h.data(), h.size() * sizeof(V), cudaMemcpyHostToDevice));
    return TOMO_OK;
}
// upload a double vector converted to the plan's arithmetic type
static int upload_real(tomo_plan *pl, void **ptr, const std::vector<double> &h) {
    if (pl->elem == 8) { double *d = nullptr; int rc = upload<double>(pl, &d, h); *ptr = d; return rc; }
    std::vector<float> hf(h.begin(), h.end());
    float *d = nullptr;
    int rc = upload<float>(pl, &d, hf);
    *ptr = d;
    return rc;
}
static int upload_twiddles(tomo_plan *pl, void **ptr, int P) {
    std::vector<double> t(2 * (size_t)P);
    for (int i = 0; i < P; ++i) { t[2 * i] = std::cos(2.0 * M_PI * i / P); t[2 * i + 1] = -std::sin(2.0 * M_PI * i / P); }
    return upload_real(pl, ptr, t);
}
}  // namespace tomo

using namespace tomo;

extern "C" const char *tomo_last_error(void) { return g_err.c_str(); }

namespace tomo {
void persist_destroy(tomo_plan *pl);
int persist_prepare_plan(tomo_plan *pl);
}

extern "C" void tomo_plan_destroy(tomo_plan *pl) {
    if (!pl) return;
    persist_destroy(pl);
    for (auto &kv : pl->graphs) cudaGraphExecDestroy(kv.second);
    for (void *p : pl->allocs) cudaFree(p);
    delete pl;
}

extern "C" int tomo_plan_create(const tomo_geometry *geom, const tomo_cn2 *cn2, double r0, double L0,
                                const tomo_noise *noise, const tomo_options *opt_in, tomo_plan **out) {
    if (!out) { set_error("out is NULL"); return TOMO_EINVAL; }
    *out = nullptr;
    tomo_options opt;
    std::memset(&opt, 0, sizeof(opt));
    opt.max_batch = 1; opt.build_cos = 1;
    if (opt_in) opt = *opt_in;
    if (opt.max_batch < 1) opt.max_batch = 1;
    if (opt.precision < TOMO_F32 || opt.precision > TOMO_F64) { set_error("unknown precision"); return TOMO_EINVAL; }
    if (opt.solver != TOMO_SOLVER_MULTIKERNEL && opt.solver != TOMO_SOLVER_PERSISTENT) { set_error("unknown solver"); return TOMO_EINVAL; }
    tomo_plan *pl = new (std::nothrow) tomo_plan();
    if (!pl) { set_error("out of host memory"); return TOMO_ENOMEM; }
    std::string err;
    int rc = build_model(geom, cn2, r0, L0, noise, opt.slope_model, opt.pad, opt.pad_os, pl->m, err, opt.layered, opt.fov_radius);
    if (rc) { set_error(err); delete pl; return rc; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) {
        set_error("no CUDA device: libtomo_b200 has no CPU fallback");
        delete pl; return TOMO_ECUDA;
    }
    cudaGetDevice(&pl->device);
    pl->opt = opt;
    pl->F = opt.max_batch;
    pl->elem = (opt.precision == TOMO_F32) ? 4 : 8;
    pl->selem = (opt.precision == TOMO_F64) ? 8 : 4;
    pl->has_cos = opt.build_cos && pl->m.T > 0;
    const HostModel &m = pl->m;
    plan_fft(m.P, pl->fd);
    plan_fft(m.P_os, pl->fd_os);

#define TRY(x) do { rc = (x); if (rc) { tomo_plan_destroy(pl); return rc; } } while (0)
    TRY(upload<int>(pl, &pl->d_row_ptr, m.row_ptr));
    TRY(upload<int>(pl, &pl->d_ix, m.ix));
    TRY(upload<int>(pl, &pl->d_iy, m.iy));
    TRY(upload<int>(pl, &pl->d_pix, m.pix));
    TRY(upload<int>(pl, &pl->d_piy, m.piy));
    TRY(upload<int>(pl, &pl->d_n_remove, m.n_remove));
    TRY(upload<int>(pl, &pl->d_interp_i0, m.interp_i0));
    TRY(upload<double>(pl, &pl->d_Gs, m.Gs));
    TRY(upload<double>(pl, &pl->d_Gphi, m.Gphi));
    TRY(upload_real(pl, &pl->d_sigma2, m.sigma2_full));
    if (!m.sigma_xy.empty()) TRY(upload_real(pl, &pl->d_sigma_xy, m.sigma_xy));
    TRY(upload_real(pl, &pl->d_interp_w, m.interp_w));
    TRY(upload_twiddles(pl, &pl->d_tw, m.P));
    TRY(upload_twiddles(pl, &pl->d_tw_os, m.P_os));

    DevGeom &g = pl->g;
    g.n = m.n; g.C = m.C; g.N = m.n_wfs; g.nv = m.nv; g.nvp = m.nvp; g.T = m.T; g.Kp = m.Kp; g.n_p = m.n_p;
    g.npairs = (m.n + 1) / 2; g.d = m.d;
    g.row_ptr = pl->d_row_ptr; g.ix = pl->d_ix; g.iy = pl->d_iy; g.pix = pl->d_pix; g.piy = pl->d_piy;
    g.n_remove = pl->d_n_remove; g.Gs = pl->d_Gs; g.Gphi = pl->d_Gphi; g.n_remove_phase = m.n_remove_phase;

    const size_t F = pl->F, vec = F * m.C * m.nv, E = pl->elem;
    TRY(dev_alloc_bytes(pl, &pl->d_x, vec * E));
    TRY(dev_alloc_bytes(pl, &pl->d_r, vec * E));
    TRY(dev_alloc_bytes(pl, &pl->d_p, vec * E));
    TRY(dev_alloc_bytes(pl, &pl->d_q, vec * E));
    TRY(dev_alloc_bytes(pl, &pl->d_b, vec * E));
    const size_t tsz = F * m.C * m.Ph * m.n * 2 * E;
    TRY(dev_alloc_bytes(pl, &pl->d_T1, tsz));
    TRY(dev_alloc_bytes(pl, &pl->d_T2, tsz));
    pl->upd_blocks = (int)std::min<size_t>(((size_t)m.C * m.nv + 255) / 256, 128);
    pl->part_stride = std::max(pl->upd_blocks, m.n_wfs);
    pl->hist_cap = 1025;
    TRY(dev_alloc<double>(pl, &pl->d_partials_q, F * m.C * g.npairs * TOMO_NRED));
    TRY(dev_alloc<double>(pl, &pl->d_partials_r, F * pl->part_stride));
    TRY(dev_alloc<double>(pl, &pl->d_hist, F * pl->hist_cap));
    TRY(dev_alloc<double>(pl, &pl->d_alpha, F + 4));
    TRY(dev_alloc_bytes(pl, &pl->d_spec, (size_t)m.Ph * m.n_pair * m.P * 2 * pl->selem));
    if (pl->has_cos) {
        // frames per projection chunk: keep the per-chunk workspaces under ~1 GiB
        const size_t per_frame = ((size_t)m.T * m.Kp * m.Ph_os * m.n_p * 2 + (size_t)m.T * m.Kp * m.n_p * m.n_p +
                                  (size_t)m.Ph_os * m.C * m.P_os * 2 + (size_t)m.C * m.Ph_os * m.n * 2) * E;
        pl->Fc = (int)std::max<size_t>(1, std::min<size_t>(F, ((size_t)1 << 30) / std::max<size_t>(per_frame, 1)));
        const size_t Fc = pl->Fc;
        TRY(dev_alloc_bytes(pl, &pl->d_z, vec * E));
        TRY(dev_alloc_bytes(pl, &pl->d_T1os, Fc * m.C * m.Ph_os * m.n * 2 * E));
        TRY(dev_alloc_bytes(pl, &pl->d_Zs, Fc * m.Ph_os * m.C * m.P_os * 2 * E));
        TRY(dev_alloc_bytes(pl, &pl->d_T2os, Fc * m.T * m.Kp * m.Ph_os * m.n_p * 2 * E));
        TRY(dev_alloc_bytes(pl, &pl->d_G, Fc * m.T * m.Kp * m.n_p * m.n_p * E));
        TRY(dev_alloc_bytes(pl, &pl->d_phi, F * m.T * m.nvp * E));
        TRY(dev_alloc<float>(pl, &pl->d_out, F * m.out_len));
        TRY(dev_alloc_bytes(pl, &pl->d_spec_os, (size_t)m.T * m.Kp * m.Ph_os * m.C * m.P_os * 2 * pl->selem));
    }
#undef TRY
    *out = pl;
    return TOMO_OK;
}

// ------------------------------------------------------------------------------------------------ upload
template <typename S>
static void pack_spectrum(const std::complex<double> *src, S *dst, size_t count) {
    for (size_t e = 0; e < count; ++e) { dst[2 * e] = (S)src[e].real(); dst[2 * e + 1] = (S)src[e].imag(); }
}

template <typename S>
static int upload_kernels_impl(tomo_plan *pl, const double *css_gen, const double *cos_gen) {
    const HostModel &m = pl->m;
    const int C = m.C, P = m.P, Ph = m.Ph, n = m.n, L = 2 * n - 1;
    {
        std::vector<double> gen_own;
        const double *gen = css_gen;
        if (!gen) { build_css_generators(m, gen_own); gen = gen_own.data(); }
        std::vector<S> host((size_t)Ph * m.n_pair * P * 2);
#pragma omp parallel
        {
            std::vector<std::complex<double>> sp((size_t)Ph * P);
#pragma omp for schedule(dynamic)
            for (int pi = 0; pi < m.n_pair; ++pi) {
                int co = 0, rem = pi;
                while (rem >= C - co) { rem -= C - co; ++co; }
                const int ci = co + rem;
                generator_spectrum(gen + ((size_t)co * C + ci) * L * L, n, n, P, sp.data());
                for (int kx = 0; kx < Ph; ++kx)
                    pack_spectrum<S>(&sp[(size_t)kx * P], &host[(((size_t)kx * m.n_pair) + pi) * P * 2], P);
            }
        }
        CK(cudaMemcpy(pl->d_spec, host.data(), host.size() * sizeof(S), cudaMemcpyHostToDevice));
    }
    if (pl->has_cos) {
        const int Po = m.P_os, Pho = m.Ph_os, Los = m.n_p + n - 1, Kp = m.Kp;
        const size_t per_t = (size_t)Kp * Pho * C * Po * 2;
        std::vector<S> host(per_t);
        for (int t = 0; t < m.T; ++t) {
            std::vector<double> gen_own;
            const double *gen = cos_gen ? cos_gen + (size_t)t * Kp * C * Los * Los : nullptr;
            if (!gen) { build_cos_generators(m, t, gen_own); gen = gen_own.data(); }
#pragma omp parallel
            {
                std::vector<std::complex<double>> sp((size_t)Pho * Po);
#pragma omp for schedule(dynamic)
                for (int kc = 0; kc < Kp * C; ++kc) {
                    const int k = kc / C, c = kc - k * C;
                    generator_spectrum(gen + (size_t)kc * Los * Los, m.n_p, n, Po, sp.data());
                    for (int kx = 0; kx < Pho; ++kx)
                        pack_spectrum<S>(&sp[(size_t)kx * Po], &host[((((size_t)k * Pho) + kx) * C + c) * Po * 2], Po);
                }
            }
            CK(cudaMemcpy((S *)pl->d_spec_os + (size_t)t * per_t, host.data(), per_t * sizeof(S), cudaMemcpyHostToDevice));
        }
    }
    pl->ready = true;
    return TOMO_OK;
}

extern "C" int tomo_plan_upload_kernels(tomo_plan *pl, const double *css_gen, const double *cos_gen) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    CK(cudaSetDevice(pl->device));
    int rc = pl->selem == 8 ? upload_kernels_impl<double>(pl, css_gen, cos_gen) : upload_kernels_impl<float>(pl, css_gen, cos_gen);
    if (rc) return rc;
    // which solver runs this plan is decided HERE, once (never inside a solve): the persistent kernel where it applies,
    // else the multi-kernel solver, with the reason kept for tomo_get_solver
    pl->solver_used = TOMO_SOLVER_MULTIKERNEL;
    pl->solver_note.clear();
    if (pl->opt.solver == TOMO_SOLVER_PERSISTENT) {
        rc = persist_prepare_plan(pl);
        if (rc == TOMO_OK) pl->solver_used = TOMO_SOLVER_PERSISTENT;
        else if (rc == TOMO_EUNSUPPORTED) pl->solver_note = g_err;
        else return rc;
    }
    return TOMO_OK;
}

// ------------------------------------------------------------------------------------------------ launch sequences
namespace tomo {

template <typename T> static Stage<T> make_stage(const tomo_plan *pl, bool os) {
    Stage<T> st;
    st.fd = os ? pl->fd_os : pl->fd;
    st.P = os ? pl->m.P_os : pl->m.P;
    st.Ph = st.P / 2 + 1;
    st.tw = reinterpret_cast<const typename cx_of<T>::type *>(os ? pl->d_tw_os : pl->d_tw);
    return st;
}

static const int kRowWarps = 4;            // warps per CTA of the row kernels (one row pair per warp)
static const int kMaxSmem = 227 * 1024;

template <typename T> static size_t rows_smem(int P) { return (size_t)(1 + 2 * kRowWarps) * P * 2 * sizeof(T); }
template <typename T> static size_t cols_smem(int P, int C, int nw) { return (size_t)(1 + 2 * C + nw) * P * 2 * sizeof(T); }
static int cols_warps(int C) { return C < 16 ? C : 16; }
static int grid_for(int items, int per_cta) { return std::max(1, std::min((items + per_cta - 1) / per_cta, 148 * 16)); }

#define LAUNCH_CHECK()                                                                     \
    do {                                                                                   \
        cudaError_t e_ = cudaGetLastError();                                               \
        if (e_ != cudaSuccess) { set_error(std::string("kernel launch: ") + cudaGetErrorString(e_)); return TOMO_ECUDA; } \
    } while (0)

static inline void prof_mark(tomo_plan *pl, cudaStream_t st) {
    if (!pl->prof) return;
    cudaEvent_t e;
    cudaEventCreate(&e);
    cudaEventRecord(e, st);
    pl->prof->push_back(e);
}

// Instantiated solve graphs are kept per (frames, iterations, flags).  The cache is bounded: a caller that sweeps many
// iteration counts on one plan would otherwise keep every graph alive; at the cap all are destroyed and rebuilt on demand
// (a graph still in flight on a stream finishes first: cudaGraphExecDestroy defers the release).
static const size_t kMaxGraphs = 32;
static inline void graph_cache_make_room(tomo_plan *pl) {
    if (pl->graphs.size() < kMaxGraphs) return;
    for (auto &kv : pl->graphs) cudaGraphExecDestroy(kv.second);
    pl->graphs.clear();
    pl->graph_launches.clear();
}

template <typename T, typename S> struct Ops {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;

    // opt in to > 48 KB of dynamic shared memory where a size needs it
    static int prepare(tomo_plan *pl) {
        const HostModel &m = pl->m;
        const size_t rs = std::max(rows_smem<T>(m.P), rows_smem<T>(m.P_os));
        const size_t cs = cols_smem<T>(m.P, m.C, cols_warps(m.C));
        if (rs > (size_t)kMaxSmem || cs > (size_t)kMaxSmem) { set_error("problem too large for the shared-memory FFT kernels"); return TOMO_EUNSUPPORTED; }
        CK(cudaFuncSetAttribute(k_rows_fwd<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs));
        CK(cudaFuncSetAttribute(k_rows_inv<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs));
        CK(cudaFuncSetAttribute(k_cos_cols_fwd<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs));
        CK(cudaFuncSetAttribute(k_cos_rows_inv<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs));
        CK(cudaFuncSetAttribute((k_cos_mac_inv<T, S>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)rs));
        CK(cudaFuncSetAttribute((k_cols<T, S>), cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cs));
        if constexpr (std::is_same<T, float>::value && std::is_same<S, float>::value) {
            const int ns = cos_bulk_stages(pl);
            if (ns > 0) {
                const int sm = (int)cos_bulk_smem(m.C, m.P_os, ns);
                switch (m.C) {
                    case 4: CK(cudaFuncSetAttribute(k_cos_mac_bulk<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm)); break;
                    case 6: CK(cudaFuncSetAttribute(k_cos_mac_bulk<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm)); break;
                    case 8: CK(cudaFuncSetAttribute(k_cos_mac_bulk<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm)); break;
                    case 12: CK(cudaFuncSetAttribute(k_cos_mac_bulk<12>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm)); break;
                    default: CK(cudaFuncSetAttribute(k_cos_mac_bulk<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, sm)); break;
                }
            }
        }
        return TOMO_OK;
    }

    // stages of the bulk-copy ring of k_cos_mac_bulk (two CTAs per SM), 0 = the kernel does not apply to this plan
    static int cos_bulk_stages(const tomo_plan *pl) {
        if (!(std::is_same<T, float>::value && std::is_same<S, float>::value)) return 0;
        const HostModel &m = pl->m;
        if (!pl->has_cos || m.P_os > kCosBulkThreads) return 0;
        if (m.C != 4 && m.C != 6 && m.C != 8 && m.C != 12 && m.C != 16) return 0;
        int ns = 0;
        while (ns < kCosBulkMaxStages && cos_bulk_smem(m.C, m.P_os, ns + 1) <= (size_t)112 * 1024) ++ns;
        return ns >= 2 ? ns : 0;
    }

    // W (Sigma_ss + Sigma_eta) W^T p -> q (modes not removed) + reduction partials; p optionally updated first
    static int mvm(tomo_plan *pl, cudaStream_t st, int F, int update, int record, int k, int n_part) {
        const HostModel &m = pl->m;
        RowsFwdArgs<T> a;
        a.st = make_stage<T>(pl, false); a.g = pl->g; a.F = F;
        a.p = (T *)pl->d_p; a.r = (const T *)pl->d_r; a.T1 = (C2 *)pl->d_T1;
        a.update = update; a.record = record; a.k = k; a.hist_stride = pl->hist_cap;
        a.partials_r = pl->d_partials_r; a.n_part = n_part; a.part_stride = pl->part_stride;
        a.hist = pl->d_hist; a.alpha = pl->d_alpha;
        const int items = F * m.C * pl->g.npairs;
        prof_mark(pl, st);
        k_rows_fwd<T><<<grid_for(items, kRowWarps), 32 * kRowWarps, rows_smem<T>(m.P), st>>>(a);
        LAUNCH_CHECK();
        prof_mark(pl, st);
        ColsArgs<T, S> c;
        c.st = a.st; c.g = pl->g; c.T1 = (const C2 *)pl->d_T1; c.T2 = (C2 *)pl->d_T2;
        c.spec = (const S2 *)pl->d_spec; c.n_pair = m.n_pair;
        const int nw = cols_warps(m.C);
        k_cols<T, S><<<dim3(m.Ph, F), 32 * nw, cols_smem<T>(m.P, m.C, nw), st>>>(c);
        LAUNCH_CHECK();
        prof_mark(pl, st);
        RowsInvArgs<T> b;
        b.st = a.st; b.g = pl->g; b.F = F; b.T2 = (const C2 *)pl->d_T2; b.p = (const T *)pl->d_p;
        b.sigma2 = (const T *)pl->d_sigma2; b.sigma_xy = (const T *)pl->d_sigma_xy; b.q = (T *)pl->d_q; b.partials_q = pl->d_partials_q;
        k_rows_inv<T><<<grid_for(items, kRowWarps), 32 * kRowWarps, rows_smem<T>(m.P), st>>>(b);
        LAUNCH_CHECK();
        prof_mark(pl, st);
        pl->launches_last += 3;
        return TOMO_OK;
    }

    static UpdateArgs<T> update_args(tomo_plan *pl, int k) {
        UpdateArgs<T> u;
        u.g = pl->g; u.x = (T *)pl->d_x; u.r = (T *)pl->d_r; u.p = (const T *)pl->d_p; u.q = (const T *)pl->d_q;
        u.partials_q = pl->d_partials_q; u.hist = pl->d_hist; u.hist_stride = pl->hist_cap; u.k = k;
        u.alpha = pl->d_alpha; u.partials_r = pl->d_partials_r; u.part_stride = pl->part_stride;
        return u;
    }

    // A7-A8 from zeta in d_z (already M_s-projected) -> d_out
    static int project_targets(tomo_plan *pl, cudaStream_t st, int F) {
        const HostModel &m = pl->m;
        const Stage<T> so = make_stage<T>(pl, true);
        const size_t rs = rows_smem<T>(m.P_os);
        for (int f0 = 0; f0 < F; f0 += pl->Fc) {
            const int Fn = std::min(pl->Fc, F - f0);
            RowsFwdArgs<T> a;
            std::memset(&a, 0, sizeof(a));
            a.st = so; a.g = pl->g; a.F = Fn; a.p = (T *)pl->d_z + (size_t)f0 * m.C * m.nv; a.r = nullptr;
            a.T1 = (C2 *)pl->d_T1os;
            k_rows_fwd<T><<<grid_for(Fn * m.C * pl->g.npairs, kRowWarps), 32 * kRowWarps, rs, st>>>(a);
            LAUNCH_CHECK();
            CosColsArgs<T> c;
            c.st = so; c.g = pl->g; c.F = Fn; c.T1 = (const C2 *)pl->d_T1os; c.Zs = (C2 *)pl->d_Zs;
            k_cos_cols_fwd<T><<<grid_for(Fn * m.C * m.Ph_os, kRowWarps), 32 * kRowWarps, rs, st>>>(c);
            LAUNCH_CHECK();
            CosMacArgs<T, S> mm;
            mm.st = so; mm.g = pl->g; mm.F = Fn; mm.Zs = (const C2 *)pl->d_Zs; mm.spec = (const S2 *)pl->d_spec_os;
            mm.T2 = (C2 *)pl->d_T2os;
            int ns = 0;
            if (Fn == 1 && (ns = cos_bulk_stages(pl)) > 0) {       // one frame, fp32: the spectra stream through a bulk-copy ring
                if constexpr (std::is_same<T, float>::value && std::is_same<S, float>::value) {
                    const int grid = std::min(2 * 148, m.T * m.Kp * m.Ph_os);
                    const size_t sm = cos_bulk_smem(m.C, m.P_os, ns);
                    switch (m.C) {
                        case 4: k_cos_mac_bulk<4><<<grid, kCosBulkThreads, sm, st>>>(mm, ns); break;
                        case 6: k_cos_mac_bulk<6><<<grid, kCosBulkThreads, sm, st>>>(mm, ns); break;
                        case 8: k_cos_mac_bulk<8><<<grid, kCosBulkThreads, sm, st>>>(mm, ns); break;
                        case 12: k_cos_mac_bulk<12><<<grid, kCosBulkThreads, sm, st>>>(mm, ns); break;
                        default: k_cos_mac_bulk<16><<<grid, kCosBulkThreads, sm, st>>>(mm, ns); break;
                    }
                }
            } else {
                k_cos_mac_inv<T, S><<<grid_for(m.T * m.Kp * m.Ph_os, kRowWarps), 32 * kRowWarps, rs, st>>>(mm);
            }
            LAUNCH_CHECK();
            CosRowsArgs<T> r;
            r.st = so; r.g = pl->g; r.F = Fn; r.T2 = (const C2 *)pl->d_T2os; r.G = (T *)pl->d_G;
            k_cos_rows_inv<T><<<grid_for(Fn * m.T * m.Kp * ((m.n_p + 1) / 2), kRowWarps), 32 * kRowWarps, rs, st>>>(r);
            LAUNCH_CHECK();
            if (m.layered) {        // L199: the layer grids ARE the result -- no I'_k, no sum over layers, no W_phi / M_phi
                const size_t cnt = (size_t)Fn * m.out_len;
                k_convert<T, float><<<(unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8), 256, 0, st>>>(
                    (const T *)pl->d_G, pl->d_out + (size_t)f0 * m.out_len, cnt);
                LAUNCH_CHECK();
                pl->launches_last += 5;
                continue;
            }
            const size_t total = (size_t)Fn * m.T * m.nvp;
            k_cos_gather<T><<<(unsigned)std::min<size_t>((total * 8 + 255) / 256, 148 * 8), 256, 0, st>>>(
                pl->g, Fn, (const T *)pl->d_G, pl->d_interp_i0, (const T *)pl->d_interp_w,
                (T *)pl->d_phi + (size_t)f0 * m.T * m.nvp);
            LAUNCH_CHECK();
            pl->launches_last += 5;
        }
        if (m.layered) return TOMO_OK;
        k_phase_project<T><<<dim3(m.T, F), 1024, 0, st>>>(pl->g, (const T *)pl->d_phi, pl->d_out);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        return TOMO_OK;
    }

    // n_iter CG iterations on the plan-held state (A2-A6), rho_{n_iter}, then the projection (A7-A8)
    static int enqueue_loop(tomo_plan *pl, cudaStream_t st, int F, int n_iter, int n_part0, bool with_cos) {
        int rc;
        for (int k = 0; k < n_iter; ++k) {
            if ((rc = mvm(pl, st, F, k > 0, 1, k, k == 0 ? n_part0 : pl->upd_blocks))) return rc;
            k_update<T><<<dim3(pl->upd_blocks, F), 256, 0, st>>>(update_args(pl, k));
            LAUNCH_CHECK();
            prof_mark(pl, st);
            pl->launches_last += 1;
        }
        k_finalize<<<F, 32, 0, st>>>(pl->d_partials_r, n_iter == 0 ? n_part0 : pl->upd_blocks, pl->part_stride,
                                     pl->d_hist, pl->hist_cap, n_iter);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        if (with_cos) {
            ProjectArgs<T, T> pa;
            pa.g = pl->g; pa.in = (const T *)pl->d_x; pa.out = (T *)pl->d_z; pa.out2 = pa.out3 = pa.zero = nullptr;
            pa.partials_r = nullptr; pa.part_stride = 0;
            k_project<T, T><<<dim3(pl->m.n_wfs, F), 1024, 0, st>>>(pa);
            LAUNCH_CHECK();
            pl->launches_last += 1;
            if ((rc = project_targets(pl, st, F))) return rc;
        }
        return TOMO_OK;
    }

    static int solve(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st) {
        const HostModel &m = pl->m;
        int rc;
        if ((rc = prepare(pl))) return rc;
        pl->launches_last = 0;
        const bool with_cos = pl->has_cos && out != nullptr;
        // A1: b = M_s s; cold start x = 0, r = p = b, rho_0 = b.b  (Eq.33-34)
        ProjectArgs<float, T> pa;
        pa.g = pl->g; pa.in = slopes; pa.out = (T *)pl->d_b; pa.out2 = (T *)pl->d_r; pa.out3 = (T *)pl->d_p;
        pa.zero = (T *)pl->d_x; pa.partials_r = pl->d_partials_r; pa.part_stride = pl->part_stride;
        k_project<float, T><<<dim3(m.n_wfs, F), 1024, 0, st>>>(pa);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        int n_part0 = m.n_wfs;
        if (x0) {   // warm start (L428, L506): r = b - A x0
            const size_t cnt = (size_t)F * m.C * m.nv;
            const unsigned gb = (unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8);
            k_convert<float, T><<<gb, 256, 0, st>>>(x0, (T *)pl->d_x, cnt);
            k_convert<float, T><<<gb, 256, 0, st>>>(x0, (T *)pl->d_p, cnt);
            LAUNCH_CHECK();
            if ((rc = mvm(pl, st, F, 0, 0, 0, 0))) return rc;
            k_warm_residual<T><<<dim3(pl->upd_blocks, F), 256, 0, st>>>(update_args(pl, 0), (const T *)pl->d_b, (T *)pl->d_p);
            LAUNCH_CHECK();
            pl->launches_last += 3;
            n_part0 = pl->upd_blocks;
        }
        {
            const auto key = std::make_tuple(F, n_iter, (x0 ? 1 : 0) + (with_cos ? 2 : 0));
            auto it = pl->graphs.find(key);
            const int before = pl->launches_last;
            if (it == pl->graphs.end()) {
                graph_cache_make_room(pl);
                cudaStream_t cs;
                CK(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
                CK(cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal));
                rc = enqueue_loop(pl, cs, F, n_iter, n_part0, with_cos);
                cudaGraph_t graph = nullptr;
                cudaError_t e = cudaStreamEndCapture(cs, &graph);
                cudaStreamDestroy(cs);
                if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
                if (e != cudaSuccess) { set_error(std::string("graph capture: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
                cudaGraphExec_t exec = nullptr;
                e = cudaGraphInstantiate(&exec, graph, 0);
                cudaGraphDestroy(graph);
                if (e != cudaSuccess) { set_error(std::string("graph instantiate: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
                it = pl->graphs.emplace(key, exec).first;
                pl->graph_launches[key] = pl->launches_last - before;
            } else {
                pl->launches_last += pl->graph_launches[key];
            }
            CK(cudaGraphLaunch(it->second, st));
        }
        if (with_cos)
            CK(cudaMemcpyAsync(out, pl->d_out, (size_t)F * m.out_len * sizeof(float), cudaMemcpyDeviceToDevice, st));
        pl->last_frames = F; pl->last_iter = n_iter;
        return TOMO_OK;
    }

    // ---- MINRES (the paper's solver for the Toeplitz method, S2.G L337, L426): same product kernels, Lanczos + Givens updates
    static MinresArgs<T> minres_args(tomo_plan *pl, int F, int k, int n_part) {
        MinresArgs<T> a;
        a.g = pl->g; a.x = (T *)pl->d_x; a.v = (T *)pl->d_p; a.v_old = (T *)pl->d_vold; a.u = (T *)pl->d_r;
        a.w1 = (T *)pl->d_w1; a.w2 = (T *)pl->d_w2; a.q = (const T *)pl->d_q; a.partials_q = pl->d_partials_q;
        a.partials_r = pl->d_partials_r; a.n_part = n_part; a.part_stride = pl->part_stride; a.state = pl->d_mstate;
        a.alpha = pl->d_alpha; a.hist = pl->d_hist; a.hist_stride = pl->hist_cap; a.k = k; a.F = F;
        return a;
    }

    static int enqueue_minres(tomo_plan *pl, cudaStream_t st, int F, int n_iter, int n_part0, bool with_cos) {
        int rc;
        const dim3 grid(pl->upd_blocks, F);
        k_minres_init<T><<<grid, 256, 0, st>>>(minres_args(pl, F, 0, n_part0));
        LAUNCH_CHECK();
        pl->launches_last += 1;
        for (int k = 0; k < n_iter; ++k) {
            if ((rc = mvm(pl, st, F, 0, 0, 0, 0))) return rc;
            k_minres_lanczos<T><<<grid, 256, 0, st>>>(minres_args(pl, F, k, pl->upd_blocks));
            k_minres_update<T><<<grid, 256, 0, st>>>(minres_args(pl, F, k, pl->upd_blocks));
            LAUNCH_CHECK();
            pl->launches_last += 2;
        }
        if (with_cos) {
            ProjectArgs<T, T> pa;
            pa.g = pl->g; pa.in = (const T *)pl->d_x; pa.out = (T *)pl->d_z; pa.out2 = pa.out3 = pa.zero = nullptr;
            pa.partials_r = nullptr; pa.part_stride = 0;
            k_project<T, T><<<dim3(pl->m.n_wfs, F), 1024, 0, st>>>(pa);
            LAUNCH_CHECK();
            pl->launches_last += 1;
            if ((rc = project_targets(pl, st, F))) return rc;
        }
        return TOMO_OK;
    }

    static int solve_minres(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st) {
        const HostModel &m = pl->m;
        int rc;
        if ((rc = prepare(pl))) return rc;
        {   // allocated on the first MINRES solve; each buffer on its own check, so a retry after a failure allocates none twice
            const size_t vec = (size_t)pl->F * m.C * m.nv * pl->elem;
            if (!pl->d_vold && (rc = dev_alloc_bytes(pl, &pl->d_vold, vec))) return rc;
            if (!pl->d_w1 && (rc = dev_alloc_bytes(pl, &pl->d_w1, vec))) return rc;
            if (!pl->d_w2 && (rc = dev_alloc_bytes(pl, &pl->d_w2, vec))) return rc;
            if (!pl->d_mstate && (rc = dev_alloc<double>(pl, &pl->d_mstate, (size_t)2 * pl->F * MS_N))) return rc;
        }
        pl->launches_last = 0;
        const bool with_cos = pl->has_cos && out != nullptr;
        // A1: b = M_s s -> d_b and d_r (the r0 of a cold start), x = 0, partial b.b  (Eq.33-34)
        ProjectArgs<float, T> pa;
        pa.g = pl->g; pa.in = slopes; pa.out = (T *)pl->d_b; pa.out2 = (T *)pl->d_r; pa.out3 = nullptr;
        pa.zero = (T *)pl->d_x; pa.partials_r = pl->d_partials_r; pa.part_stride = pl->part_stride;
        k_project<float, T><<<dim3(m.n_wfs, F), 1024, 0, st>>>(pa);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        int n_part0 = m.n_wfs;
        if (x0) {   // warm start (L428, L506): r0 = b - A x0
            const size_t cnt = (size_t)F * m.C * m.nv;
            const unsigned gb = (unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8);
            k_convert<float, T><<<gb, 256, 0, st>>>(x0, (T *)pl->d_x, cnt);
            k_convert<float, T><<<gb, 256, 0, st>>>(x0, (T *)pl->d_p, cnt);
            LAUNCH_CHECK();
            if ((rc = mvm(pl, st, F, 0, 0, 0, 0))) return rc;
            k_warm_residual<T><<<dim3(pl->upd_blocks, F), 256, 0, st>>>(update_args(pl, 0), (const T *)pl->d_b, (T *)pl->d_p);
            LAUNCH_CHECK();
            pl->launches_last += 3;
            n_part0 = pl->upd_blocks;
        }
        const auto key = std::make_tuple(F, n_iter, 4 + (x0 ? 1 : 0) + (with_cos ? 2 : 0));
        auto it = pl->graphs.find(key);
        const int before = pl->launches_last;
        if (it == pl->graphs.end()) {
            graph_cache_make_room(pl);
            cudaStream_t cs;
            CK(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
            CK(cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal));
            rc = enqueue_minres(pl, cs, F, n_iter, n_part0, with_cos);
            cudaGraph_t graph = nullptr;
            cudaError_t e = cudaStreamEndCapture(cs, &graph);
            cudaStreamDestroy(cs);
            if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
            if (e != cudaSuccess) { set_error(std::string("graph capture: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
            cudaGraphExec_t exec = nullptr;
            e = cudaGraphInstantiate(&exec, graph, 0);
            cudaGraphDestroy(graph);
            if (e != cudaSuccess) { set_error(std::string("graph instantiate: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
            it = pl->graphs.emplace(key, exec).first;
            pl->graph_launches[key] = pl->launches_last - before;
        } else {
            pl->launches_last += pl->graph_launches[key];
        }
        CK(cudaGraphLaunch(it->second, st));
        if (with_cos)
            CK(cudaMemcpyAsync(out, pl->d_out, (size_t)F * m.out_len * sizeof(float), cudaMemcpyDeviceToDevice, st));
        pl->last_frames = F; pl->last_iter = n_iter;
        return TOMO_OK;
    }

    static int apply_css(tomo_plan *pl, const float *v, float *out, cudaStream_t st) {
        int rc;
        if ((rc = prepare(pl))) return rc;
        pl->launches_last = 0;
        ProjectArgs<float, T> pa;
        pa.g = pl->g; pa.in = v; pa.out = (T *)pl->d_p; pa.out2 = pa.out3 = pa.zero = nullptr; pa.partials_r = nullptr; pa.part_stride = 0;
        k_project<float, T><<<dim3(pl->m.n_wfs, 1), 256, 0, st>>>(pa);
        LAUNCH_CHECK();
        if ((rc = mvm(pl, st, 1, 0, 0, 0, 0))) return rc;
        ProjectArgs<T, float> pb;
        pb.g = pl->g; pb.in = (const T *)pl->d_q; pb.out = out; pb.out2 = pb.out3 = pb.zero = nullptr; pb.partials_r = nullptr; pb.part_stride = 0;
        k_project<T, float><<<dim3(pl->m.n_wfs, 1), 256, 0, st>>>(pb);
        LAUNCH_CHECK();
        pl->launches_last += 2;
        return TOMO_OK;
    }

    // tomo_apply_css_static: the multi-kernel product of apply_css with every workspace inside the caller-given scratch
    // (layout p | q | T1 | T2 | partials_q, each part 256-byte aligned); returns the bytes needed in *need
    static size_t static_layout(const tomo_plan *pl, size_t off[5]) {
        const HostModel &m = pl->m;
        const size_t vec = (size_t)m.C * m.nv * sizeof(T), tsz = (size_t)m.C * m.Ph * m.n * 2 * sizeof(T);
        const size_t sz[5] = {vec, vec, tsz, tsz, (size_t)m.C * pl->g.npairs * TOMO_NRED * sizeof(double)};
        size_t o = 0;
        for (int i = 0; i < 5; ++i) { off[i] = o; o += (sz[i] + 255) & ~(size_t)255; }
        return o;
    }
    static int apply_css_static(tomo_plan *pl, const float *v, float *out, cudaStream_t st, unsigned char *scr, size_t cap) {
        const HostModel &m = pl->m;
        size_t off[5];
        const size_t need = static_layout(pl, off);
        if (need > cap) {
            set_error("tomo_apply_css_static: this plan needs " + std::to_string(need) + " bytes of workspace, the static scratch holds " +
                      std::to_string(cap) + " (TOMO_STATIC_SCRATCH_BYTES); use tomo_apply_css");
            return TOMO_EINVAL;
        }
        int rc;
        if ((rc = prepare(pl))) return rc;
        T *sp = (T *)(scr + off[0]), *sq = (T *)(scr + off[1]);
        C2 *t1 = (C2 *)(scr + off[2]), *t2 = (C2 *)(scr + off[3]);
        double *part = (double *)(scr + off[4]);
        // the array keeps the last call's contents (possibly another plan's): cleared, so that no call ever sees them
        CK(cudaMemsetAsync(scr, 0, need, st));
        ProjectArgs<float, T> pa;
        pa.g = pl->g; pa.in = v; pa.out = sp; pa.out2 = pa.out3 = pa.zero = nullptr; pa.partials_r = nullptr; pa.part_stride = 0;
        k_project<float, T><<<dim3(m.n_wfs, 1), 256, 0, st>>>(pa);
        LAUNCH_CHECK();
        RowsFwdArgs<T> a;
        std::memset(&a, 0, sizeof(a));
        a.st = make_stage<T>(pl, false); a.g = pl->g; a.F = 1; a.p = sp; a.T1 = t1;
        const int items = m.C * pl->g.npairs;
        k_rows_fwd<T><<<grid_for(items, kRowWarps), 32 * kRowWarps, rows_smem<T>(m.P), st>>>(a);
        LAUNCH_CHECK();
        ColsArgs<T, S> c;
        c.st = a.st; c.g = pl->g; c.T1 = t1; c.T2 = t2; c.spec = (const S2 *)pl->d_spec; c.n_pair = m.n_pair;
        const int nw = cols_warps(m.C);
        k_cols<T, S><<<dim3(m.Ph, 1), 32 * nw, cols_smem<T>(m.P, m.C, nw), st>>>(c);
        LAUNCH_CHECK();
        RowsInvArgs<T> b;
        b.st = a.st; b.g = pl->g; b.F = 1; b.T2 = t2; b.p = sp;
        b.sigma2 = (const T *)pl->d_sigma2; b.sigma_xy = (const T *)pl->d_sigma_xy; b.q = sq; b.partials_q = part;
        k_rows_inv<T><<<grid_for(items, kRowWarps), 32 * kRowWarps, rows_smem<T>(m.P), st>>>(b);
        LAUNCH_CHECK();
        ProjectArgs<T, float> pb;
        pb.g = pl->g; pb.in = sq; pb.out = out; pb.out2 = pb.out3 = pb.zero = nullptr; pb.partials_r = nullptr; pb.part_stride = 0;
        k_project<T, float><<<dim3(m.n_wfs, 1), 256, 0, st>>>(pb);
        LAUNCH_CHECK();
        return TOMO_OK;
    }

    static int apply_cos(tomo_plan *pl, const float *zeta, float *out, cudaStream_t st) {
        int rc;
        if ((rc = prepare(pl))) return rc;
        pl->launches_last = 0;
        ProjectArgs<float, T> pa;
        pa.g = pl->g; pa.in = zeta; pa.out = (T *)pl->d_z; pa.out2 = pa.out3 = pa.zero = nullptr; pa.partials_r = nullptr; pa.part_stride = 0;
        k_project<float, T><<<dim3(pl->m.n_wfs, 1), 256, 0, st>>>(pa);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        if ((rc = project_targets(pl, st, 1))) return rc;
        CK(cudaMemcpyAsync(out, pl->d_out, pl->m.out_len * sizeof(float), cudaMemcpyDeviceToDevice, st));
        return TOMO_OK;
    }

    static int cg_step(tomo_plan *pl, float *x, float *r, float *p, double *scal, cudaStream_t st) {
        int rc;
        if ((rc = prepare(pl))) return rc;
        pl->launches_last = 0;
        const size_t cnt = (size_t)pl->m.C * pl->m.nv;
        const unsigned gb = (unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8);
        k_convert<float, T><<<gb, 256, 0, st>>>(x, (T *)pl->d_x, cnt);
        k_convert<float, T><<<gb, 256, 0, st>>>(r, (T *)pl->d_r, cnt);
        k_convert<float, T><<<gb, 256, 0, st>>>(p, (T *)pl->d_p, cnt);
        LAUNCH_CHECK();
        CK(cudaMemcpyAsync(pl->d_hist, scal, sizeof(double), cudaMemcpyDeviceToDevice, st));
        if ((rc = mvm(pl, st, 1, 0, 0, 0, 0))) return rc;
        k_update<T><<<dim3(pl->upd_blocks, 1), 256, 0, st>>>(update_args(pl, 0));
        LAUNCH_CHECK();
        k_step_finish<T><<<gb, 256, 0, st>>>(pl->g, (const T *)pl->d_r, (T *)pl->d_p, pl->d_partials_r, pl->upd_blocks,
                                             pl->d_hist, pl->d_alpha, scal);
        LAUNCH_CHECK();
        k_convert<T, float><<<gb, 256, 0, st>>>((const T *)pl->d_x, x, cnt);
        k_convert<T, float><<<gb, 256, 0, st>>>((const T *)pl->d_r, r, cnt);
        k_convert<T, float><<<gb, 256, 0, st>>>((const T *)pl->d_p, p, cnt);
        LAUNCH_CHECK();
        pl->launches_last += 8;
        return TOMO_OK;
    }

    // one un-graphed pass of the iteration loop on the plan-held state with an event after every kernel
    static int time_kernels(tomo_plan *pl, int F, int n_iter, float *ms_out, cudaStream_t st) {
        int rc;
        if ((rc = prepare(pl))) return rc;
        std::vector<cudaEvent_t> ev;
        pl->prof = &ev;
        rc = enqueue_loop(pl, st, F, n_iter, pl->upd_blocks, false);
        pl->prof = nullptr;
        cudaError_t e = cudaStreamSynchronize(st);
        double acc[4] = {0, 0, 0, 0};
        if (!rc && e == cudaSuccess && (int)ev.size() == 5 * n_iter)
            for (int k = 0; k < n_iter; ++k)
                for (int j = 0; j < 4; ++j) {
                    float ms = 0.f;
                    cudaEventElapsedTime(&ms, ev[5 * k + j], ev[5 * k + j + 1]);
                    acc[j] += ms;
                }
        else if (!rc) { set_error("profiling pass failed"); rc = TOMO_ECUDA; }
        for (cudaEvent_t x : ev) cudaEventDestroy(x);
        for (int j = 0; j < 4; ++j) ms_out[j] = (float)(acc[j] / std::max(n_iter, 1));
        return rc;
    }

    // A7-A8 after the persistent solver: the seven small kernels are replayed from one CUDA graph per frame count (their
    // arguments are plan-owned buffers), which shortens the gaps between the dependent launches
    static int project_from_x(tomo_plan *pl, cudaStream_t st, int F) {
        int rc;
        if ((rc = prepare(pl))) return rc;
        {
            const auto key = std::make_tuple(F, -1, 8);
            auto it = pl->graphs.find(key);
            if (it == pl->graphs.end()) {
                graph_cache_make_room(pl);
                const int before = pl->launches_last;
                cudaStream_t cs;
                CK(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
                CK(cudaStreamBeginCapture(cs, cudaStreamCaptureModeThreadLocal));
                rc = project_from_x_enqueue(pl, cs, F);
                cudaGraph_t graph = nullptr;
                cudaError_t e = cudaStreamEndCapture(cs, &graph);
                cudaStreamDestroy(cs);
                if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
                if (e != cudaSuccess) { set_error(std::string("graph capture: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
                cudaGraphExec_t exec = nullptr;
                e = cudaGraphInstantiate(&exec, graph, 0);
                cudaGraphDestroy(graph);
                if (e != cudaSuccess) { set_error(std::string("graph instantiate: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
                it = pl->graphs.emplace(key, exec).first;
                pl->graph_launches[key] = pl->launches_last - before;
            } else {
                pl->launches_last += pl->graph_launches[key];
            }
            CK(cudaGraphLaunch(it->second, st));
            return TOMO_OK;
        }
    }

    static int project_from_x_enqueue(tomo_plan *pl, cudaStream_t st, int F) {
        ProjectArgs<T, T> pa;
        pa.g = pl->g; pa.in = (const T *)pl->d_x; pa.out = (T *)pl->d_z; pa.out2 = pa.out3 = pa.zero = nullptr;
        pa.partials_r = nullptr; pa.part_stride = 0;
        k_project<T, T><<<dim3(pl->m.n_wfs, F), 1024, 0, st>>>(pa);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        return project_targets(pl, st, F);
    }

    static int state_load(tomo_plan *pl, cudaStream_t st, const float *x, const float *r, const float *p, const double *rho) {
        const size_t cnt = (size_t)pl->m.C * pl->m.nv;
        const unsigned gb = (unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8);
        k_convert<float, T><<<gb, 256, 0, st>>>(x, (T *)pl->d_x, cnt);
        k_convert<float, T><<<gb, 256, 0, st>>>(r, (T *)pl->d_r, cnt);
        k_convert<float, T><<<gb, 256, 0, st>>>(p, (T *)pl->d_p, cnt);
        LAUNCH_CHECK();
        CK(cudaMemcpyAsync(pl->d_hist, rho, sizeof(double), cudaMemcpyDeviceToDevice, st));
        pl->launches_last += 3;
        return TOMO_OK;
    }

    static int state_store(tomo_plan *pl, cudaStream_t st, float *x, float *r, float *p) {
        const size_t cnt = (size_t)pl->m.C * pl->m.nv;
        const unsigned gb = (unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8);
        k_convert<T, float><<<gb, 256, 0, st>>>((const T *)pl->d_x, x, cnt);
        k_convert<T, float><<<gb, 256, 0, st>>>((const T *)pl->d_r, r, cnt);
        k_convert<T, float><<<gb, 256, 0, st>>>((const T *)pl->d_p, p, cnt);
        LAUNCH_CHECK();
        pl->launches_last += 3;
        return TOMO_OK;
    }

    static int vec_store(tomo_plan *pl, cudaStream_t st, const void *src, float *dst) {
        const size_t cnt = (size_t)pl->m.C * pl->m.nv;
        k_convert<T, float><<<(unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8), 256, 0, st>>>((const T *)src, dst, cnt);
        LAUNCH_CHECK();
        pl->launches_last += 1;
        return TOMO_OK;
    }

    static int get_zeta(tomo_plan *pl, float *out, int F, cudaStream_t st) {
        const size_t cnt = (size_t)F * pl->m.C * pl->m.nv;
        k_convert<T, float><<<(unsigned)std::min<size_t>((cnt + 255) / 256, 148 * 8), 256, 0, st>>>((const T *)pl->d_x, out, cnt);
        LAUNCH_CHECK();
        return TOMO_OK;
    }
};
}  // namespace tomo

// ------------------------------------------------------------------------------------------------ ABI entry points
#define DISPATCH(pl, CALL)                                                       \
    ((pl)->opt.precision == TOMO_F32 ? Ops<float, float>::CALL                   \
     : (pl)->opt.precision == TOMO_F32S_F64A ? Ops<double, float>::CALL : Ops<double, double>::CALL)

static int check_ready(tomo_plan *pl) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    if (!pl->ready) { set_error("tomo_plan_upload_kernels has not been called"); return TOMO_ENOTREADY; }
    cudaError_t e = cudaSetDevice(pl->device);
    if (e != cudaSuccess) { set_error(std::string("cudaSetDevice: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    return TOMO_OK;
}

namespace tomo {
int solve_persistent(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st);
int cg_step_persistent(tomo_plan *pl, float *x, float *r, float *p, double *scal, cudaStream_t st);
int time_phases_persistent(tomo_plan *pl, int F, int n_iter, int minres, float *us_out, cudaStream_t st);
int time_solver_persistent(tomo_plan *pl, const float *slopes, int F, int n_iter, int reps, int minres, float *ms_out, cudaStream_t st);

// A7-A8 from the CG solution held in d_x -> d_out (used by the persistent solver)
int project_from_x(tomo_plan *pl, cudaStream_t st, int F) { return DISPATCH(pl, project_from_x(pl, st, F)); }
// fp32 ABI vectors <-> plan-held CG state (teacher-forced step)
int state_load(tomo_plan *pl, cudaStream_t st, const float *x, const float *r, const float *p, const double *rho) {
    return DISPATCH(pl, state_load(pl, st, x, r, p, rho));
}
int state_store(tomo_plan *pl, cudaStream_t st, float *x, float *r, float *p) { return DISPATCH(pl, state_store(pl, st, x, r, p)); }
int vec_store(tomo_plan *pl, cudaStream_t st, const void *src, float *dst) { return DISPATCH(pl, vec_store(pl, st, src, dst)); }
int apply_css_persistent(tomo_plan *pl, const float *v, float *out, cudaStream_t st);
int solve_minres_persistent(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st);
}  // namespace tomo

extern "C" int tomo_solve_batch(tomo_plan *pl, const float *slopes, float *wavefront_out, int n_frames, int n_iter,
                                const float *x0, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!slopes) { set_error("slopes is NULL"); return TOMO_EINVAL; }
    if (n_frames < 1 || n_frames > pl->F) { set_error("n_frames outside [1, max_batch]"); return TOMO_EINVAL; }
    if (n_iter < 0 || n_iter >= pl->hist_cap) { set_error("n_iter outside [0, 1024]"); return TOMO_EINVAL; }
    if (pl->has_cos && !wavefront_out) { set_error("wavefront_out is NULL"); return TOMO_EINVAL; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    if (pl->solver_used == TOMO_SOLVER_PERSISTENT) return solve_persistent(pl, slopes, wavefront_out, n_frames, n_iter, x0, st);
    return DISPATCH(pl, solve(pl, slopes, wavefront_out, n_frames, n_iter, x0, st));
}

extern "C" int tomo_solve_minres(tomo_plan *pl, const float *slopes, float *wavefront_out, int n_frames, int n_iter,
                                 const float *x0, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!slopes) { set_error("slopes is NULL"); return TOMO_EINVAL; }
    if (n_frames < 1 || n_frames > pl->F) { set_error("n_frames outside [1, max_batch]"); return TOMO_EINVAL; }
    if (n_iter < 0 || n_iter >= pl->hist_cap) { set_error("n_iter outside [0, 1024]"); return TOMO_EINVAL; }
    if (pl->has_cos && !wavefront_out) { set_error("wavefront_out is NULL"); return TOMO_EINVAL; }
    if (pl->solver_used == TOMO_SOLVER_PERSISTENT) return solve_minres_persistent(pl, slopes, wavefront_out, n_frames, n_iter, x0, (cudaStream_t)cuda_stream);
    return DISPATCH(pl, solve_minres(pl, slopes, wavefront_out, n_frames, n_iter, x0, (cudaStream_t)cuda_stream));
}

extern "C" int tomo_solve(tomo_plan *pl, const float *slopes, float *wavefront_out, int n_iter, void *cuda_stream) {
    return tomo_solve_batch(pl, slopes, wavefront_out, 1, n_iter, nullptr, cuda_stream);
}

extern "C" int tomo_apply_css(tomo_plan *pl, const float *v, float *out, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!v || !out) { set_error("NULL vector"); return TOMO_EINVAL; }
    // the product of the solver that runs the solves: one single-product launch of the persistent kernel, or the multi-kernel product
    if (pl->solver_used == TOMO_SOLVER_PERSISTENT) return apply_css_persistent(pl, v, out, (cudaStream_t)cuda_stream);
    return DISPATCH(pl, apply_css(pl, v, out, (cudaStream_t)cuda_stream));
}

// ---- the product without any allocation (tomo.h: tomo_apply_css_static).  The workspace is this file-scope device array: every
// GPU that loads the library holds TOMO_STATIC_SCRATCH_BYTES of it until the process exits.  In host code the name below is a
// host-side stand-in, not a device address: the address is asked for once per device, with that device current.
static __device__ __align__(256) unsigned char g_static_scratch[TOMO_STATIC_SCRATCH_BYTES];
static std::mutex g_static_mu;
static unsigned char *g_static_ptr[64] = {};

static int static_scratch_address(int device, unsigned char **out) {
    if (device < 0 || device >= 64) { set_error("tomo_apply_css_static: device index out of range"); return TOMO_EUNSUPPORTED; }
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[device]) {
        void *ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_static_scratch);        // the caller made `device` current (check_ready)
        if (e != cudaSuccess || !ptr) { set_error(std::string("cudaGetSymbolAddress(g_static_scratch): ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
        g_static_ptr[device] = (unsigned char *)ptr;
    }
    *out = g_static_ptr[device];
    return TOMO_OK;
}

extern "C" int tomo_apply_css_static(tomo_plan *pl, const float *v, float *out, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!v || !out) { set_error("NULL vector"); return TOMO_EINVAL; }
    unsigned char *scr = nullptr;
    if ((rc = static_scratch_address(pl->device, &scr))) return rc;
    return DISPATCH(pl, apply_css_static(pl, v, out, (cudaStream_t)cuda_stream, scr, (size_t)TOMO_STATIC_SCRATCH_BYTES));
}

extern "C" int tomo_apply_cos(tomo_plan *pl, const float *zeta, float *wavefront_out, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!pl->has_cos) { set_error("plan was created without the target projection"); return TOMO_EINVAL; }
    if (!zeta || !wavefront_out) { set_error("NULL vector"); return TOMO_EINVAL; }
    return DISPATCH(pl, apply_cos(pl, zeta, wavefront_out, (cudaStream_t)cuda_stream));
}

extern "C" int tomo_cg_step(tomo_plan *pl, float *x, float *r, float *p, double *rho_alpha_beta, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!x || !r || !p || !rho_alpha_beta) { set_error("NULL vector"); return TOMO_EINVAL; }
    if (pl->solver_used == TOMO_SOLVER_PERSISTENT) return cg_step_persistent(pl, x, r, p, rho_alpha_beta, (cudaStream_t)cuda_stream);
    return DISPATCH(pl, cg_step(pl, x, r, p, rho_alpha_beta, (cudaStream_t)cuda_stream));
}

extern "C" int tomo_get_zeta(tomo_plan *pl, float *zeta_out, int n_frames, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!zeta_out || n_frames < 1 || n_frames > pl->F) { set_error("bad arguments"); return TOMO_EINVAL; }
    return DISPATCH(pl, get_zeta(pl, zeta_out, n_frames, (cudaStream_t)cuda_stream));
}

extern "C" int tomo_time_kernels(tomo_plan *pl, int n_frames, int n_iter, float *ms_out, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!ms_out || n_frames < 1 || n_frames > pl->F || n_iter < 1 || n_iter >= pl->hist_cap) { set_error("bad arguments"); return TOMO_EINVAL; }
    return DISPATCH(pl, time_kernels(pl, n_frames, n_iter, ms_out, (cudaStream_t)cuda_stream));
}

extern "C" int tomo_time_phases(tomo_plan *pl, int n_frames, int n_iter, int minres, float *us_out, void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!us_out || n_frames < 1 || n_frames > pl->F || n_iter < 1 || n_iter >= pl->hist_cap) { set_error("bad arguments"); return TOMO_EINVAL; }
    return time_phases_persistent(pl, n_frames, n_iter, minres, us_out, (cudaStream_t)cuda_stream);
}

extern "C" int tomo_time_solver(tomo_plan *pl, const float *slopes, int n_frames, int n_iter, int reps, int minres, float *ms_out,
                                void *cuda_stream) {
    int rc = check_ready(pl);
    if (rc) return rc;
    if (!slopes || !ms_out || n_frames < 1 || n_frames > pl->F || n_iter < 0 || n_iter >= pl->hist_cap || reps < 1 || reps > 10000) {
        set_error("bad arguments");
        return TOMO_EINVAL;
    }
    return time_solver_persistent(pl, slopes, n_frames, n_iter, reps, minres, ms_out, (cudaStream_t)cuda_stream);
}

// ---- measurement aid: L2 read bandwidth and fp32 FMA rate of the device (tomo_measure_device)
namespace tomo {
__global__ void __launch_bounds__(256) k_l2_sweep(const float4 *buf, size_t n4, int sweeps, float *sink) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (int s = 0; s < sweeps; ++s)
        for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n4; i += 4 * stride) {
            // four independent 16-byte L2 loads in flight per thread
            const float4 a = __ldcg(buf + i);
            const float4 b = (i + stride < n4) ? __ldcg(buf + i + stride) : make_float4(0.f, 0.f, 0.f, 0.f);
            const float4 c = (i + 2 * stride < n4) ? __ldcg(buf + i + 2 * stride) : make_float4(0.f, 0.f, 0.f, 0.f);
            const float4 d = (i + 3 * stride < n4) ? __ldcg(buf + i + 3 * stride) : make_float4(0.f, 0.f, 0.f, 0.f);
            acc.x += a.x + b.x + c.x + d.x; acc.y += a.y + b.y + c.y + d.y;
            acc.z += a.z + b.z + c.z + d.z; acc.w += a.w + b.w + c.w + d.w;
        }
    if (acc.x + acc.y + acc.z + acc.w == 12345.678f) sink[0] = acc.x;      // keeps the loads alive
}
__global__ void __launch_bounds__(256) k_fma_rate(int iters, float *sink) {
    float a[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) a[j] = 1.0f + 1e-3f * (threadIdx.x + j);
    const float m = 0.999f, c = 1e-3f;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int j = 0; j < 8; ++j) a[j] = fmaf(a[j], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += a[j];
    if (s == 12345.678f) sink[0] = s;
}
}  // namespace tomo

extern "C" int tomo_measure_device(long long l2_bytes, int reps, float *out, void *cuda_stream) {
    if (!out || reps < 1 || reps > 1000 || l2_bytes < 0) { set_error("bad arguments"); return TOMO_EINVAL; }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { set_error("no CUDA device: libtomo_b200 has no CPU fallback"); return TOMO_ECUDA; }
    cudaStream_t st = (cudaStream_t)cuda_stream;
    int dev = 0, sms = 0;
    CK(cudaGetDevice(&dev));
    CK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const size_t bytes = l2_bytes ? (size_t)l2_bytes : ((size_t)64 << 20);
    const size_t n4 = bytes / 16;
    float4 *buf = nullptr;
    float *sink = nullptr;
    CK(cudaMalloc(&buf, n4 * 16));
    if (cudaMalloc(&sink, 16) != cudaSuccess || cudaMemsetAsync(buf, 0, n4 * 16, st) != cudaSuccess) {
        set_error(std::string("tomo_measure_device: ") + cudaGetErrorString(cudaGetLastError()));
        cudaFree(buf); cudaFree(sink);
        return TOMO_ECUDA;
    }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    const int sweeps = 20;
    float best_bw = 0.f, best_fl = 0.f;
    k_l2_sweep<<<sms * 8, 256, 0, st>>>(buf, n4, 2, sink);             // warm: the buffer becomes L2-resident
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0, st);
        k_l2_sweep<<<sms * 8, 256, 0, st>>>(buf, n4, sweeps, sink);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms > 0.f) best_bw = std::max(best_bw, (float)((double)n4 * 16 * sweeps / (ms * 1e-3) / 1e9));
    }
    const int iters = 20000;
    for (int r = 0; r < reps; ++r) {
        cudaEventRecord(e0, st);
        k_fma_rate<<<sms * 8, 256, 0, st>>>(iters, sink);
        cudaEventRecord(e1, st);
        if (cudaEventSynchronize(e1) != cudaSuccess) break;
        float ms = 0.f;
        cudaEventElapsedTime(&ms, e0, e1);
        if (ms > 0.f) best_fl = std::max(best_fl, (float)((double)sms * 8 * 256 * iters * 8 * 2 / (ms * 1e-3) / 1e12));
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaError_t e = cudaGetLastError();
    cudaFree(buf); cudaFree(sink);
    if (e != cudaSuccess) { set_error(std::string("tomo_measure_device: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    out[0] = best_bw; out[1] = best_fl;
    return TOMO_OK;
}

extern "C" int tomo_get_sizes(const tomo_plan *pl, int *n_vs, int *n_vphi, int *slopes_len, int *wavefront_len,
                              int *pad, int *pad_os, int *n_prime) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    if (n_vs) *n_vs = pl->m.nv;
    if (n_vphi) *n_vphi = pl->m.layered ? pl->m.n_p * pl->m.n_p : pl->m.nvp;
    if (slopes_len) *slopes_len = pl->m.C * pl->m.nv;
    if (wavefront_len) *wavefront_len = (int)pl->m.out_len;
    if (pad) *pad = pl->m.P;
    if (pad_os) *pad_os = pl->m.P_os;
    if (n_prime) *n_prime = pl->m.n_p;
    return TOMO_OK;
}

extern "C" int tomo_get_valid_index(const tomo_plan *pl, int *subap_idx, int *phase_idx) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    if (subap_idx) std::memcpy(subap_idx, pl->m.sub_idx.data(), pl->m.sub_idx.size() * sizeof(int));
    if (phase_idx) std::memcpy(phase_idx, pl->m.ph_idx.data(), pl->m.ph_idx.size() * sizeof(int));
    return TOMO_OK;
}

extern "C" int tomo_get_noise(const tomo_plan *pl, double *sigma2_wfs, double *slope_var) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    if (sigma2_wfs) std::memcpy(sigma2_wfs, pl->m.sigma2_wfs.data(), pl->m.sigma2_wfs.size() * sizeof(double));
    if (slope_var) *slope_var = pl->m.slope_var;
    return TOMO_OK;
}

extern "C" int tomo_get_residuals(const tomo_plan *pl, double *host_out, int n_frames, int n_iter) {
    if (!pl || !host_out) { set_error("NULL argument"); return TOMO_EINVAL; }
    if (n_frames < 1 || n_frames > pl->F || n_iter < 0 || n_iter >= pl->hist_cap) { set_error("bad sizes"); return TOMO_EINVAL; }
    std::vector<double> h((size_t)n_frames * pl->hist_cap);
    CK(cudaMemcpy(h.data(), pl->d_hist, h.size() * sizeof(double), cudaMemcpyDeviceToHost));
    for (int f = 0; f < n_frames; ++f)
        for (int k = 0; k <= n_iter; ++k) host_out[(size_t)f * (n_iter + 1) + k] = std::sqrt(h[(size_t)f * pl->hist_cap + k]);
    return TOMO_OK;
}

extern "C" int tomo_get_solver(const tomo_plan *pl, int *solver_in_use, char *note, int note_cap) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    if (!pl->ready) { set_error("tomo_plan_upload_kernels has not been called"); return TOMO_ENOTREADY; }
    if (solver_in_use) *solver_in_use = pl->solver_used;
    if (note && note_cap > 0) { std::strncpy(note, pl->solver_note.c_str(), (size_t)note_cap - 1); note[note_cap - 1] = 0; }
    return TOMO_OK;
}

extern "C" int tomo_get_stats(const tomo_plan *pl, long long *device_bytes, int *launches_last_solve) {
    if (!pl) { set_error("plan is NULL"); return TOMO_EINVAL; }
    if (device_bytes) *device_bytes = (long long)pl->bytes;
    if (launches_last_solve) *launches_last_solve = pl->launches_last;
    return TOMO_OK;
}

// ------------------------------------------------------------------------------------------------ host-only builders
// (declared in include/tomo_host.h; no device needed -- used by the CPU test-suite to check row A0)
static int host_model_from(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model, int pad,
                           int pad_os, HostModel &m) {
    std::string err;
    tomo_noise nz; std::memset(&nz, 0, sizeof(nz));
    int rc = build_model(g, cn2, r0, L0, &nz, slope_model, pad, pad_os, m, err);
    if (rc) set_error(err);
    return rc;
}

extern "C" int tomo_host_sizes(const tomo_geometry *g, const tomo_cn2 *cn2, int pad, int pad_os, int *n_vs, int *n_vphi,
                               int *n_prime, int *P, int *P_os, int *Kp) {
    HostModel m;
    int rc = host_model_from(g, cn2, 0.15, 25.0, TOMO_HUDGIN, pad, pad_os, m);
    if (rc) return rc;
    if (n_vs) *n_vs = m.nv;
    if (n_vphi) *n_vphi = m.nvp;
    if (n_prime) *n_prime = m.n_p;
    if (P) *P = m.P;
    if (P_os) *P_os = m.P_os;
    if (Kp) *Kp = m.Kp;
    return TOMO_OK;
}

extern "C" int tomo_host_css_generators(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                                        double *gen_out) {
    HostModel m;
    int rc = host_model_from(g, cn2, r0, L0, slope_model, 0, 0, m);
    if (rc) return rc;
    std::vector<double> gen;
    build_css_generators(m, gen);
    std::memcpy(gen_out, gen.data(), gen.size() * sizeof(double));
    return TOMO_OK;
}

extern "C" int tomo_host_cos_generators(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                                        int target, double *gen_out) {
    HostModel m;
    int rc = host_model_from(g, cn2, r0, L0, slope_model, 0, 0, m);
    if (rc) return rc;
    if (target < 0 || target >= m.T) { set_error("target out of range"); return TOMO_EINVAL; }
    std::vector<double> gen;
    build_cos_generators(m, target, gen);
    std::memcpy(gen_out, gen.data(), gen.size() * sizeof(double));
    return TOMO_OK;
}

extern "C" int tomo_host_layer_generators(const tomo_geometry *g, const tomo_cn2 *cn2, double r0, double L0, int slope_model,
                                          double fov_radius, int *n_m_out, double *gen_out) {
    HostModel m;
    std::string err;
    tomo_noise nz; std::memset(&nz, 0, sizeof(nz));
    int rc = build_model(g, cn2, r0, L0, &nz, slope_model, 0, 0, m, err, 1, fov_radius);
    if (rc) { set_error(err); return rc; }
    if (n_m_out) *n_m_out = m.n_p;
    if (!gen_out) return TOMO_OK;
    std::vector<double> gen;
    build_cos_generators(m, 0, gen);
    std::memcpy(gen_out, gen.data(), gen.size() * sizeof(double));
    return TOMO_OK;
}

extern "C" int tomo_host_generator_spectrum(const double *gen, int n_out, int n_in, int P, double *spec_out) {
    if (!gen || !spec_out || P % 2 || !is_5smooth(P) || P < n_out + n_in - 1) { set_error("bad arguments"); return TOMO_EINVAL; }
    std::vector<std::complex<double>> sp((size_t)(P / 2 + 1) * P);
    generator_spectrum(gen, n_out, n_in, P, sp.data());
    for (size_t e = 0; e < sp.size(); ++e) { spec_out[2 * e] = sp[e].real(); spec_out[2 * e + 1] = sp[e].imag(); }
    return TOMO_OK;
}

extern "C" int tomo_host_structure_function(const double *r, int count, double r0, double L0, double *out) {
    if (!r || !out || count < 0) { set_error("bad arguments"); return TOMO_EINVAL; }
    for (int i = 0; i < count; ++i) out[i] = structure_function(r[i], r0, L0);
    return TOMO_OK;
}
