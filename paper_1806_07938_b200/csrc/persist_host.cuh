// persist_host.cuh -- host side of the persistent solver shared by solve_persistent.cu (prepare, dispatch) and the
// per-size translation units persist_inst.cu (kernel instantiation + launch).
#pragma once
#include <algorithm>
#include <cstring>
#include <set>
#include <string>
#include <type_traits>
#include <vector>

#include "tomo.h"
#include "persist_kernel.cuh"
#include "tomo_plan.hpp"

namespace tomo {

// FFT edges the persistent kernel is instantiated for (one translation unit each); other sizes use the multi-kernel solver
#define TOMO_PERSIST_SIZES(X) X(16) X(20) X(24) X(32) X(40) X(64) X(128) X(160) X(192) X(256)

struct PersistState {
    unsigned *d_flags = nullptr;
    void *d_T1 = nullptr, *d_T1p = nullptr, *d_T2 = nullptr, *d_mspec = nullptr, *d_s2c = nullptr;
    void *d_xd = nullptr, *d_rd = nullptr, *d_pd = nullptr, *d_bd = nullptr, *d_w1d = nullptr, *d_w2d = nullptr;
    double *d_part_r = nullptr, *d_part_s = nullptr, *d_part_i = nullptr;
    int G = 0, nq_m = 1, NQ = 0, NQ_mr = 0, SB = 0, any_remove = 0, spec_smem = 0, vec_smem = 0, vec_smem_mr = 0;
    int off_ms = 0, off_work = 0, off_red = 0, off_scal = 0, off_tab = 0, off_upart = 0, off_vm = 0, off_vec = 0, off_spec = 0, off_ptab = 0, off_unit = 0, ngs = 2;
    int off_ms2 = 0, fb = 1;
    size_t smem = 0;
    std::set<const void *> attr_set;    // kernel instances whose dynamic shared-memory limit has been raised
    int *d_seg = nullptr;        // [F_max + 1][sms][8] slab segment tables, one per frame count (slab_segments), uploaded by persist_prepare
    int sms = 0;
};

// balance of the Ph x F slab passes over G CTAs (persist_kernel.cuh, phase C): host table [G][8]
void slab_segments(int Ph, int F, int G, std::vector<int> &seg);

struct PLaunch {
    int F, n_iter, mode, finalize_p, method;
    const float *slopes, *x0;
    double *scal_out;
    long long *dbg;
};

#define PCK(call)                                                                 \
    do {                                                                          \
        cudaError_t e_ = (call);                                                  \
        if (e_ != cudaSuccess) {                                                  \
            set_error(std::string(#call) + ": " + cudaGetErrorString(e_));        \
            return TOMO_ECUDA;                                                    \
        }                                                                         \
    } while (0)

template <int P> int persist_run(tomo_plan *pl, cudaStream_t st, const PLaunch &L);

template <typename T, typename S, int P>
static int persist_launch(tomo_plan *pl, cudaStream_t st, const PLaunch &L) {
    typedef typename cx_of<T>::type C2;
    typedef typename cx_of<S>::type S2;
    PersistState *ps = (PersistState *)pl->persist;
    const HostModel &m = pl->m;
    PArgs<T, S> a;
    std::memset(&a, 0, sizeof(a));
    a.g = pl->g;
    a.P = m.P; a.Ph = m.Ph; a.tw = (const C2 *)pl->d_tw;
    a.F = L.F; a.n_iter = L.n_iter; a.mode = L.mode; a.finalize_p = L.finalize_p;
    a.npad = 2 * pl->g.npairs; a.U = m.C * pl->g.npairs; a.NQ = ps->NQ; a.nq_m = ps->nq_m; a.SB = ps->SB;
    a.G = std::max(1, std::min(ps->G, std::max(L.F * a.U, m.Ph)));
    a.spec_smem = ps->spec_smem; a.vec_smem = ps->vec_smem; a.any_remove = ps->any_remove;
    a.off_ms = ps->off_ms; a.off_work = ps->off_work; a.off_red = ps->off_red; a.off_scal = ps->off_scal;
    a.off_tab = ps->off_tab; a.off_upart = ps->off_upart; a.off_vm = ps->off_vm; a.off_vec = ps->off_vec;
    a.off_spec = ps->off_spec; a.off_ptab = ps->off_ptab; a.off_unit = ps->off_unit; a.ngs = ps->ngs;
    a.off_ms2 = ps->off_ms2; a.fb = ps->fb;
    a.seg = ps->d_seg + (size_t)L.F * ps->sms * 8;
    a.s_in = L.slopes; a.x0 = L.x0;
    a.x = (T *)pl->d_x; a.r = (T *)pl->d_r; a.p = (T *)pl->d_p;
    a.xd = (T *)ps->d_xd; a.rd = (T *)ps->d_rd; a.pd = (T *)ps->d_pd; a.bd = (T *)ps->d_bd;
    a.T1 = (C2 *)ps->d_T1; a.T1p = (C2 *)ps->d_T1p; a.T2 = (C2 *)ps->d_T2;
    a.spec = (const S2 *)pl->d_spec; a.n_pair = m.n_pair;
    a.mspec = (const C2 *)ps->d_mspec; a.s2c = (const T *)ps->d_s2c;
    a.part_r = ps->d_part_r; a.part_s = ps->d_part_s; a.part_i = ps->d_part_i;
    a.hist = pl->d_hist; a.hist_stride = pl->hist_cap; a.alpha = pl->d_alpha; a.scal_out = L.scal_out;
    a.flags = ps->d_flags; a.dbg = L.dbg;
    // the instrumented instances (tomo_time_phases) exist for TOMO_F32 only (MINRES: single frame); the production instances
    // carry no stamp code
    const bool mr = L.method == METHOD_MINRES;
    const void *kern = mr ? (L.F > 1 ? (const void *)(k_persistent<T, S, P, true, false, METHOD_MINRES>) : (const void *)(k_persistent<T, S, P, false, false, METHOD_MINRES>))
                          : (L.F > 1 ? (const void *)(k_persistent<T, S, P, true, false, METHOD_CG>) : (const void *)(k_persistent<T, S, P, false, false, METHOD_CG>));
    if (L.dbg) {
        if constexpr (std::is_same<T, float>::value && std::is_same<S, float>::value) {
            if (mr && L.F > 1) { set_error("tomo_time_phases: the instrumented MINRES instance runs one frame"); return TOMO_EUNSUPPORTED; }
            kern = mr ? (const void *)(k_persistent<T, S, P, false, true, METHOD_MINRES>) : L.F > 1 ? (const void *)(k_persistent<T, S, P, true, true, METHOD_CG>) : (const void *)(k_persistent<T, S, P, false, true, METHOD_CG>);
        } else { set_error("tomo_time_phases: the instrumented kernel instances exist for TOMO_F32 only"); return TOMO_EUNSUPPORTED; }
    }
    if (mr) { a.NQ = ps->NQ_mr; a.vec_smem = ps->vec_smem_mr; a.w1d = (T *)ps->d_w1d; a.w2d = (T *)ps->d_w2d; }
    if (!ps->attr_set.count(kern)) {
        PCK(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)ps->smem));
        int occ = 0;
        PCK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, kPThreads, ps->smem));
        if (occ < 1) { set_error("persistent kernel does not fit on an SM"); return TOMO_EUNSUPPORTED; }
        ps->attr_set.insert(kern);
    }
    PCK(cudaMemsetAsync(ps->d_flags, 0, 1024, st));
    void *kargs[] = {&a};
    PCK(cudaLaunchCooperativeKernel(kern, dim3(a.G), dim3(kPThreads), kargs, ps->smem, st));
    pl->launches_last += 1;
    return TOMO_OK;
}

}  // namespace tomo
