// tomo_plan.hpp -- the opaque plan behind include/tomo.h: host model + every device allocation + graph cache.
#pragma once
#include <cuda_runtime.h>

#include <map>
#include <string>
#include <tuple>
#include <vector>

#include "host_model.hpp"
#include "tomo_kernels.cuh"

struct tomo_plan {
    tomo::HostModel m;
    tomo_options opt;
    bool ready = false;          // spectra uploaded
    bool has_cos = false;
    int device = 0;
    int F = 1;                   // max_batch
    int Fc = 1;                  // frames per chunk of the target projection
    int hist_cap = 0;            // doubles per frame in d_hist
    int upd_blocks = 1;          // gridDim.x of k_update = number of r.r partials per frame
    int part_stride = 1;
    size_t elem = 4, selem = 4;  // sizeof(T), sizeof(S)
    size_t bytes = 0;
    int launches_last = 0;
    int last_frames = 0, last_iter = 0;

    tomo::DevGeom g;
    tomo::FftDesc fd, fd_os;
    // device tables
    int *d_row_ptr = nullptr, *d_ix = nullptr, *d_iy = nullptr, *d_pix = nullptr, *d_piy = nullptr,
        *d_n_remove = nullptr, *d_interp_i0 = nullptr;
    double *d_Gs = nullptr, *d_Gphi = nullptr;
    void *d_tw = nullptr, *d_tw_os = nullptr, *d_sigma2 = nullptr, *d_sigma_xy = nullptr, *d_interp_w = nullptr;
    void *d_spec = nullptr, *d_spec_os = nullptr;
    // CG state and workspaces (arithmetic type T)
    void *d_x = nullptr, *d_r = nullptr, *d_p = nullptr, *d_q = nullptr, *d_b = nullptr;
    void *d_T1 = nullptr, *d_T2 = nullptr;
    double *d_partials_q = nullptr, *d_partials_r = nullptr, *d_hist = nullptr, *d_alpha = nullptr;
    // MINRES state (allocated by the first tomo_solve_minres): v_{k-1}, w_{k-1}, w_{k-2}, rotation scalars
    void *d_vold = nullptr, *d_w1 = nullptr, *d_w2 = nullptr;
    double *d_mstate = nullptr;
    // target projection
    void *d_z = nullptr, *d_T1os = nullptr, *d_Zs = nullptr, *d_T2os = nullptr, *d_G = nullptr, *d_phi = nullptr;
    float *d_out = nullptr;      // [F][T][nvp]
    std::vector<void *> allocs;
    // graph cache: (n_frames, n_iter, warm) -> executable graph of the iteration loop + projection
    std::map<std::tuple<int, int, int>, cudaGraphExec_t> graphs;
    std::map<std::tuple<int, int, int>, int> graph_launches;   // kernel nodes in each cached graph
    std::vector<cudaEvent_t> *prof = nullptr;   // when set, launch sequences bracket every kernel with events
    void *persist = nullptr;     // persistent-solver state (solve_persistent.cu)
    int solver_used = 0;         // TOMO_SOLVER_* that actually runs the solves: decided once, in tomo_plan_upload_kernels
    std::string solver_note;     // why the persistent solver was not taken (empty when it was, or was not asked for)
};

namespace tomo {
void set_error(const std::string &s);
}
