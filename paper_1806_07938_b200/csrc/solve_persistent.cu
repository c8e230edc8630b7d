// solve_persistent.cu -- host side of the persistent cooperative CG solver (kernel: persist_kernel.cuh; one
// instantiation per FFT edge in persist_inst.cu): shared-memory layout, workspaces, dispatch, measurement aid.
#include <algorithm>
#include <complex>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "persist_host.cuh"
#include "tomo_host.h"
#include "tomo_kernels_cos.cuh"

namespace tomo {

static int palloc(tomo_plan *pl, void **ptr, size_t bytes) {
    void *p = nullptr;
    bytes = std::max<size_t>(bytes, 16);
    cudaError_t e = cudaMalloc(&p, bytes);
    if (e != cudaSuccess) { set_error(std::string("cudaMalloc: ") + cudaGetErrorString(e)); return TOMO_ENOMEM; }
    pl->allocs.push_back(p);
    pl->bytes += bytes;
    *ptr = p;
    return TOMO_OK;
}

static size_t align16(size_t v) { return (v + 15) & ~(size_t)15; }

// spectra of the pupil mask and of the coordinate-weighted masks: [nq_m][Ph][P] complex fp64
static void build_mask_spectra(const HostModel &m, int nq_m, std::vector<std::complex<double>> &out) {
    const int P = m.P, Ph = m.Ph;
    out.assign((size_t)nq_m * Ph * P, 0.0);
    std::vector<std::complex<double>> img((size_t)P * P);
    for (int q = 0; q < nq_m; ++q) {
        std::fill(img.begin(), img.end(), 0.0);
        for (int i = 0; i < m.nv; ++i) {
            double wv = 1.0;
            if (q == 1) wv = (m.ix[i] - 0.5 * (m.n - 1)) * m.d;
            if (q == 2) wv = (m.iy[i] - 0.5 * (m.n - 1)) * m.d;
            img[(size_t)m.iy[i] * P + m.ix[i]] = wv;
        }
        for (int y = 0; y < P; ++y) host_fft(&img[(size_t)y * P], P, 1, false);      // along x
        for (int x = 0; x < P; ++x) host_fft(&img[x], P, P, false);                  // along y
        for (int kx = 0; kx < Ph; ++kx)
            for (int ky = 0; ky < P; ++ky) out[((size_t)q * Ph + kx) * P + ky] = img[(size_t)ky * P + kx];
    }
}

// Balance of the slab passes of phase C.  CTA b owns slab k_x = b % Ph together with the other CTAs of that residue and
// takes an even share of the F frames (its spectra stay pinned in shared memory).  With F > 1 the slabs that have one CTA
// fewer carry up to twice the frames: those CTAs hand the frames beyond the average to CTAs below the average, which
// process them as a second, "helped" slab with the spectra read through L2.  One helped slab per CTA.
// seg[b] = {own f_lo, own f_hi, helped k_x, helped f_lo, helped f_hi, 0, 0, 0}.
void slab_segments(int Ph, int F, int G, std::vector<int> &seg) {
    seg.assign((size_t)G * 8, 0);
    std::vector<int> share(G);
    for (int b = 0; b < G; ++b) {
        const int kx = b % Ph, cnt = (G - 1 - kx) / Ph + 1, rk = b / Ph;
        int lo = (int)((long long)rk * F / cnt), hi = (int)((long long)(rk + 1) * F / cnt);
        if (F == 1) { lo = 0; hi = rk == 0 ? 1 : 0; }
        seg[b * 8 + 0] = lo; seg[b * 8 + 1] = hi; seg[b * 8 + 2] = kx;
        share[b] = hi - lo;
    }
    const int target = (int)(((long long)Ph * F + G - 1) / G);
    int h = 0;                                                   // next helper candidate
    for (int b = 0; b < G; ++b) {
        while (share[b] > target) {
            while (h < G && !(share[h] < target && seg[h * 8 + 4] == seg[h * 8 + 3])) ++h;
            if (h >= G) return;                                  // no helper left: the owner keeps the rest
            const int take = std::min(share[b] - target, target - share[h]);
            const int hi = seg[b * 8 + 1];
            seg[h * 8 + 2] = b % Ph; seg[h * 8 + 3] = hi - take; seg[h * 8 + 4] = hi;
            seg[b * 8 + 1] = hi - take;
            share[b] -= take; share[h] += take;
            ++h;
        }
    }
}

}  // namespace tomo

extern "C" int tomo_host_slab_segments(int Ph, int n_frames, int n_ctas, int *seg_out) {
    if (Ph < 1 || n_frames < 1 || n_ctas < Ph || !seg_out) { tomo::set_error("bad arguments"); return TOMO_EINVAL; }
    std::vector<int> seg;
    tomo::slab_segments(Ph, n_frames, n_ctas, seg);
    std::memcpy(seg_out, seg.data(), seg.size() * sizeof(int));
    return TOMO_OK;
}

namespace tomo {

static int persist_prepare(tomo_plan *pl) {
    if (pl->persist) return TOMO_OK;
    const HostModel &m = pl->m;
    // Sigma_eta uniform per channel?
    for (int c = 0; c < m.C; ++c)
        for (int i = 1; i < m.nv; ++i)
            if (m.sigma2_full[(size_t)c * m.nv + i] != m.sigma2_full[(size_t)c * m.nv]) {
                set_error("persistent solver needs a noise variance that is uniform per WFS channel");
                return TOMO_EUNSUPPORTED;
            }
    if (!m.sigma_xy.empty()) { set_error("persistent solver needs a diagonal noise covariance"); return TOMO_EUNSUPPORTED; }
    int dev = 0, sms = 0, coop = 0, max_smem = 0;
    PCK(cudaGetDevice(&dev));
    PCK(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    PCK(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
    PCK(cudaDeviceGetAttribute(&max_smem, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev));
    if (!coop) { set_error("device does not support cooperative launches"); return TOMO_EUNSUPPORTED; }
    int fa = 0, fb = 0;
    bool size_ok = false;
#define TOMO_PSZ(P_) size_ok = size_ok || (m.P == P_);
    TOMO_PERSIST_SIZES(TOMO_PSZ)
#undef TOMO_PSZ
    if (!size_ok || !fact2_of(m.P, &fa, &fb) || fb > kGS) { set_error("persistent solver: FFT edge not instantiated"); return TOMO_EUNSUPPORTED; }
    if (m.Ph > sms || m.Ph > 160 || sms > 160) { set_error("persistent solver: more k_x slabs than SMs (or than 160)"); return TOMO_EUNSUPPORTED; }
    if ((m.P + 31) / 32 > kPWarps || m.C * fb > kPThreads || m.C * ((m.n + 1) / 2) > 2 * kPThreads || m.n > 16 * kGS) { set_error("persistent solver: FFT edge or channel count too large"); return TOMO_EUNSUPPORTED; }
    PersistState *ps = new PersistState();
    const int npairs = (m.n + 1) / 2, U = m.C * npairs, F = pl->F;
    ps->G = std::max(1, std::min(sms, std::max(F * U, m.Ph)));
    ps->any_remove = 0;
    bool focus = false;
    for (int i = 0; i < m.n_wfs; ++i) { if (m.n_remove[i] > 0) ps->any_remove = 1; if (m.n_remove[i] > 2) focus = true; }
    ps->nq_m = focus ? 3 : 1;
    ps->NQ = 1 + m.C * (focus ? 2 : 1);
    ps->NQ_mr = 1 + 2 * m.C * (focus ? 2 : 1);            // MINRES: the modal sums of v_k too (reading G27)
    ps->SB = SC_HEAD + 4 * m.C + 3 * m.n_wfs + MR_N;       // CG block, then MINRES' sums of v and recurrence state
    const size_t E = pl->elem, SE = pl->selem;
    const int WPG = (m.P + 31) / 32, Goc = std::min(kPWarps / WPG, m.C);
    const int maxu = (F * U + ps->G - 1) / ps->G;
    const size_t LD = (size_t)fa * (fb + 1);
    // row-unit slots per round: as few rounds as 32 groups allow, then as few slots as those rounds need
    const int rounds = std::max(1, (maxu + kPThreads / kGS - 1) / (kPThreads / kGS));
    ps->ngs = std::min(kPThreads / kGS, (((maxu + rounds - 1) / rounds) + 1) & ~1);
    // frames per slab pass of the batch instance: two when the FFT passes have the threads for it AND the doubled pass buffers
    // fit (P = 256 with 16 frames: they do not, and one frame per pass keeps the plan on the persistent kernel)
    size_t off = 0;
    for (int fbp = (F > 1 && 2 * m.C * fb <= kPThreads) ? 2 : 1; fbp >= 1; --fbp) {
        ps->fb = fbp;
        off = (size_t)m.P * 2 * E;
        ps->off_ms = (int)(off = align16(off));
        off += (size_t)ps->nq_m * m.P * 2 * E;
        ps->off_ms2 = (int)(off = align16(off));
        off += (size_t)ps->nq_m * m.P * 2 * E + 32;      // + the CTA's row of the slab segment table
        ps->off_work = (int)(off = align16(off));
        off += std::max((size_t)2 * ps->fb * m.C * LD, (size_t)ps->ngs * (m.P + LD)) * 2 * E;
        ps->off_red = (int)(off = align16(off));
        off += (size_t)ps->fb * (Goc + 4 * m.C) * m.P * E;
        ps->off_scal = (int)(off = align16(off));
        off += (size_t)F * ps->SB * sizeof(double);
        ps->off_tab = (int)(off = align16(off));
        off += (size_t)m.n_wfs * (9 * sizeof(double) + sizeof(int)) + 8 + (size_t)(m.C + 2) * E + 16;
        ps->off_upart = (int)(off = align16(off));
        off += std::max((size_t)maxu * sizeof(double), (size_t)m.C * 4 * E);      // [C][4] mode coefficients (single-frame instance)
        ps->off_vm = (int)(off = align16(off));
        off += (size_t)maxu * kGS * sizeof(unsigned);
        ps->off_ptab = (int)(off = align16(off));
        off += (size_t)m.C * m.C * sizeof(PairRef);
        ps->off_unit = (int)(off = align16(off));
        off += (size_t)std::max(maxu, 1) * sizeof(UnitRec);
        off = align16(off);
        const size_t spec_bytes = (size_t)m.n_pair * m.P * 2 * SE, vec_bytes = (size_t)maxu * 6 * m.n * E, vec_bytes_mr = (size_t)maxu * 10 * m.n * E;
        // the spectra slice has priority for the shared memory that is left, then the CG vectors of the CTA's row units
        ps->off_spec = (int)off;
        ps->spec_smem = off + spec_bytes <= (size_t)max_smem;
        if (ps->spec_smem) off = align16(off + spec_bytes);
        ps->off_vec = (int)off;
        ps->vec_smem = off + vec_bytes <= (size_t)max_smem;
        ps->vec_smem_mr = ps->vec_smem && (off + vec_bytes_mr <= (size_t)max_smem);      // MINRES keeps five row vectors per unit
        if (ps->vec_smem) off = align16(off + (ps->vec_smem_mr ? vec_bytes_mr : vec_bytes));
        if (off <= (size_t)max_smem) break;
    }
    if (off > (size_t)max_smem) { delete ps; set_error("persistent solver: problem too large for shared memory"); return TOMO_EUNSUPPORTED; }
    ps->smem = off;

    int rc;
#define PTRY(x) do { rc = (x); if (rc) { delete ps; return rc; } } while (0)
    const size_t tsz = (size_t)F * m.Ph * m.C * 2 * npairs * 2 * E;
    const size_t dsz = (size_t)F * m.C * 2 * npairs * m.n * E;
    PTRY(palloc(pl, (void **)&ps->d_flags, 1024));
    ps->sms = sms;
    PTRY(palloc(pl, (void **)&ps->d_seg, (size_t)(F + 1) * sms * 8 * sizeof(int)));
    {   // slab work tables of every frame count a solve may be given: the solve path itself never synchronises with the host
        std::vector<int> all((size_t)(F + 1) * sms * 8, 0), seg;
        for (int f = 1; f <= F; ++f) {
            const int Gf = std::max(1, std::min(ps->G, std::max(f * U, m.Ph)));
            slab_segments(m.Ph, f, Gf, seg);
            std::copy(seg.begin(), seg.end(), all.begin() + (size_t)f * sms * 8);
        }
        cudaError_t e = cudaMemcpy(ps->d_seg, all.data(), all.size() * sizeof(int), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) { delete ps; set_error(std::string("cudaMemcpy: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    }
    PTRY(palloc(pl, &ps->d_T1, tsz));
    PTRY(palloc(pl, &ps->d_T1p, tsz));
    PTRY(palloc(pl, &ps->d_T2, tsz));
    PTRY(palloc(pl, &ps->d_xd, dsz));
    PTRY(palloc(pl, &ps->d_rd, dsz));
    PTRY(palloc(pl, &ps->d_pd, dsz));
    PTRY(palloc(pl, &ps->d_bd, dsz));
    PTRY(palloc(pl, (void **)&ps->d_part_r, (size_t)F * U * sizeof(double)));
    PTRY(palloc(pl, (void **)&ps->d_part_s, (size_t)F * m.Ph * ps->NQ_mr * sizeof(double)));
    if (!ps->vec_smem_mr) { PTRY(palloc(pl, &ps->d_w1d, dsz)); PTRY(palloc(pl, &ps->d_w2d, dsz)); }
    PTRY(palloc(pl, (void **)&ps->d_part_i, (size_t)F * U * 2 * sizeof(double)));
    PTRY(palloc(pl, &ps->d_mspec, (size_t)ps->nq_m * m.Ph * m.P * 2 * E));
    PTRY(palloc(pl, &ps->d_s2c, (size_t)m.C * E));
#undef PTRY
    std::vector<std::complex<double>> msp;
    build_mask_spectra(m, ps->nq_m, msp);
    std::vector<double> s2(m.C);
    for (int c = 0; c < m.C; ++c) s2[c] = m.sigma2_full[(size_t)c * m.nv] / ((double)m.P * m.P);
    if (E == 8) {
        PCK(cudaMemcpy(ps->d_mspec, msp.data(), msp.size() * 16, cudaMemcpyHostToDevice));
        PCK(cudaMemcpy(ps->d_s2c, s2.data(), s2.size() * 8, cudaMemcpyHostToDevice));
    } else {
        std::vector<float> mf(msp.size() * 2), sf(s2.begin(), s2.end());
        for (size_t i = 0; i < msp.size(); ++i) { mf[2 * i] = (float)msp[i].real(); mf[2 * i + 1] = (float)msp[i].imag(); }
        PCK(cudaMemcpy(ps->d_mspec, mf.data(), mf.size() * 4, cudaMemcpyHostToDevice));
        PCK(cudaMemcpy(ps->d_s2c, sf.data(), sf.size() * 4, cudaMemcpyHostToDevice));
    }
    pl->persist = ps;
    return TOMO_OK;
}

static int persist_dispatch(tomo_plan *pl, cudaStream_t st, int F, int n_iter, int mode, int finalize_p, const float *slopes,
                            const float *x0, double *scal_out, long long *dbg = nullptr, int method = METHOD_CG) {
    PLaunch L;
    L.F = F; L.n_iter = n_iter; L.mode = mode; L.finalize_p = finalize_p; L.slopes = slopes; L.x0 = x0; L.scal_out = scal_out; L.dbg = dbg;
    L.method = method;
    switch (pl->m.P) {
#define TOMO_PCASE(P_) case P_: return persist_run<P_>(pl, st, L);
        TOMO_PERSIST_SIZES(TOMO_PCASE)
#undef TOMO_PCASE
        default: break;
    }
    set_error("persistent solver: FFT edge not instantiated");
    return TOMO_EUNSUPPORTED;
}

int project_from_x(tomo_plan *pl, cudaStream_t st, int F);       // tomo_api.cu: A7-A8 from d_x -> d_out
int state_load(tomo_plan *pl, cudaStream_t st, const float *x, const float *r, const float *p, const double *rho);
int state_store(tomo_plan *pl, cudaStream_t st, float *x, float *r, float *p);

int solve_persistent(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    pl->launches_last = 0;
    if ((rc = persist_dispatch(pl, st, F, n_iter, x0 ? PM_WARM : PM_COLD, 0, slopes, x0, nullptr))) return rc;
    if (pl->has_cos && out) {
        if ((rc = project_from_x(pl, st, F))) return rc;
        PCK(cudaMemcpyAsync(out, pl->d_out, (size_t)F * pl->m.out_len * sizeof(float), cudaMemcpyDeviceToDevice, st));
    }
    pl->last_frames = F; pl->last_iter = n_iter;
    return TOMO_OK;
}

// MINRES (the paper's solver for the Toeplitz method, L337, L426) inside the persistent kernel: same phases, same two exchanges
// per iteration as CG (persist_kernel.cuh: METHOD_MINRES)
int solve_minres_persistent(tomo_plan *pl, const float *slopes, float *out, int F, int n_iter, const float *x0, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    pl->launches_last = 0;
    if ((rc = persist_dispatch(pl, st, F, n_iter, x0 ? PM_WARM : PM_COLD, 0, slopes, x0, nullptr, nullptr, METHOD_MINRES))) return rc;
    if (pl->has_cos && out) {
        if ((rc = project_from_x(pl, st, F))) return rc;
        PCK(cudaMemcpyAsync(out, pl->d_out, (size_t)F * pl->m.out_len * sizeof(float), cudaMemcpyDeviceToDevice, st));
    }
    pl->last_frames = F; pl->last_iter = n_iter;
    return TOMO_OK;
}

// one product through the persistent kernel (tomo_apply_css with the persistent solver): r <- M_s (W Sigma_ss W^T + Sigma_eta) M_s^T v
int vec_store(tomo_plan *pl, cudaStream_t st, const void *src, float *dst);
int apply_css_persistent(tomo_plan *pl, const float *v, float *out, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    pl->launches_last = 0;
    if ((rc = persist_dispatch(pl, st, 1, 1, PM_APPLY, 0, v, nullptr, nullptr))) return rc;
    return vec_store(pl, st, pl->d_r, out);
}

// decided once, when the spectra are uploaded: can the persistent solver run this plan?  (TOMO_EUNSUPPORTED = no)
int persist_prepare_plan(tomo_plan *pl) { return persist_prepare(pl); }

// one teacher-forced iteration through the persistent kernel (tomo_cg_step with the persistent solver)
int cg_step_persistent(tomo_plan *pl, float *x, float *r, float *p, double *scal, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    pl->launches_last = 0;
    if ((rc = state_load(pl, st, x, r, p, scal))) return rc;
    if ((rc = persist_dispatch(pl, st, 1, 1, PM_STATE, 1, nullptr, nullptr, scal))) return rc;
    return state_store(pl, st, x, r, p);
}

// Measurement aid (tomo_time_phases): one instrumented persistent solve -- CG from the state the last solve left
// (PM_STATE), MINRES from a cold start on the projected slopes the last solve left in the plan -- thread 0 of every CTA stamps clock64 at the phase boundaries; returns, per segment, the mean over
// iterations of the MAXIMUM over CTAs (work segments) or the MINIMUM over CTAs (barrier waits = pure latency).
int time_phases_persistent(tomo_plan *pl, int F, int n_iter, int minres, float *us_out, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    PersistState *ps = (PersistState *)pl->persist;
    const int G = std::max(1, std::min(ps->G, std::max(F * pl->m.C * pl->g.npairs, pl->m.Ph)));
    long long *d_dbg = nullptr;
    const size_t cnt = (size_t)G * n_iter * PT_N;
    PCK(cudaMalloc(&d_dbg, cnt * sizeof(long long)));
    PCK(cudaMemsetAsync(d_dbg, 0, cnt * sizeof(long long), st));
    if (minres && pl->elem != 4) { cudaFree(d_dbg); set_error("tomo_time_phases: MINRES is instrumented for TOMO_F32 only"); return TOMO_EUNSUPPORTED; }
    rc = minres ? persist_dispatch(pl, st, F, n_iter, PM_COLD, 0, (const float *)pl->d_b, nullptr, nullptr, d_dbg, METHOD_MINRES)
                : persist_dispatch(pl, st, F, n_iter, PM_STATE, 0, nullptr, nullptr, nullptr, d_dbg);
    std::vector<long long> h(cnt);
    cudaError_t e = cudaStreamSynchronize(st);
    if (!rc && e == cudaSuccess) e = cudaMemcpy(h.data(), d_dbg, cnt * sizeof(long long), cudaMemcpyDeviceToHost);
    cudaFree(d_dbg);
    if (rc) return rc;
    if (e != cudaSuccess) { set_error(std::string("time_phases: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, pl->device);
    const double us_per_cycle = 1e3 / std::max(khz, 1);
    // optional raw timeline: per CTA, mean over iterations of every stamp relative to the iteration start [us]
    if (const char *path = getenv("TOMO_STAMP_DUMP")) {
        if (FILE *fp = fopen(path, "w")) {
            for (int b = 0; b < G; ++b) {
                fprintf(fp, "%d", b);
                for (int s = 0; s < PT_N; ++s) {
                    double acc = 0.0;
                    for (int k = 0; k < n_iter; ++k) {
                        const long long *t = &h[((size_t)b * n_iter + k) * PT_N];
                        acc += t[s] ? (double)(t[s] - t[PT_START]) : 0.0;
                    }
                    fprintf(fp, " %.3f", acc * us_per_cycle / n_iter);
                }
                fprintf(fp, "\n");
            }
            fclose(fp);
        }
    }
    const int n_seg = PT_BAR_A + 1;                   // the ten segments of the ABI (tomo_time_phases)
    for (int s = 0; s < n_seg; ++s) us_out[s] = 0.f;
    for (int k = 0; k < n_iter; ++k)
        for (int s = 1; s < n_seg; ++s) {
            const bool wait = (s == PT_BAR_B || s == PT_BAR_A);
            const bool slab_seg = (s >= PT_BUILD && s <= PT_INV);
            long long best = wait ? (1LL << 62) : 0;
            for (int b = 0; b < G; ++b) {
                const long long *t = &h[((size_t)b * n_iter + k) * PT_N];
                const bool has_slab = t[PT_MAC] != 0;
                if (slab_seg && !has_slab) continue;
                if (s == PT_BAR_B && !has_slab) continue;
                const long long prev = (s == PT_BAR_B && !has_slab) ? t[PT_RHO] : t[s - 1];
                const long long dt = t[s] - prev;
                best = wait ? std::min(best, dt) : std::max(best, dt);
            }
            us_out[s] += (float)(best * us_per_cycle / n_iter);
        }
    // total per iteration as seen by CTA 0
    us_out[0] = n_iter > 1 ? (float)((h[((size_t)(n_iter - 1)) * PT_N + PT_BAR_A] - h[PT_START]) * us_per_cycle / n_iter) : 0.f;
    return TOMO_OK;
}

// Measurement aid (tomo_time_solver): the persistent kernel alone, `reps` cold-start launches bracketed by events.
int time_solver_persistent(tomo_plan *pl, const float *slopes, int F, int n_iter, int reps, int minres, float *ms_out, cudaStream_t st) {
    int rc;
    if ((rc = persist_prepare(pl))) return rc;
    std::vector<cudaEvent_t> ev(2 * (size_t)reps);
    for (auto &e : ev) PCK(cudaEventCreate(&e));
    for (int i = 0; i < reps && !rc; ++i) {
        PersistState *ps = (PersistState *)pl->persist;
        PCK(cudaMemsetAsync(ps->d_flags, 0, 1024, st));     // (the launch below repeats it; keeps the bracket tight)
        PCK(cudaEventRecord(ev[2 * i], st));
        rc = persist_dispatch(pl, st, F, n_iter, PM_COLD, 0, slopes, nullptr, nullptr, nullptr, minres ? METHOD_MINRES : METHOD_CG);
        PCK(cudaEventRecord(ev[2 * i + 1], st));
    }
    cudaError_t e = cudaStreamSynchronize(st);
    double tot = 0.0;
    for (int i = 0; i < reps; ++i) { float ms = 0.f; cudaEventElapsedTime(&ms, ev[2 * i], ev[2 * i + 1]); tot += ms; }
    for (auto &x : ev) cudaEventDestroy(x);
    if (rc) return rc;
    if (e != cudaSuccess) { set_error(std::string("time_solver: ") + cudaGetErrorString(e)); return TOMO_ECUDA; }
    *ms_out = (float)(tot / reps);
    return TOMO_OK;
}

void persist_destroy(tomo_plan *pl) {
    delete (PersistState *)pl->persist;
    pl->persist = nullptr;
}

}  // namespace tomo
