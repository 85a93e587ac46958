// kernels.h -- host-callable launchers of libacm's CUDA kernels.  Each kernel family lives in its
// own translation unit (phase_*.cu, hydro_*.cu, aux.cu, ...) so that the library builds in
// parallel; the launchers dispatch the runtime (stencil, walls, storage state, variant) tuple to
// the matching template instance and enqueue it on the given stream.  They return the
// cudaGetLastError() of the launch.
#pragma once
#include "common.cuh"

namespace acm {

struct Launch {
    dim3 grid, block;
    cudaStream_t stream;
};

// Fused phase-field LB step (one launch).  state = storage state the kernel reads.
template <typename T> cudaError_t launch_phase(int Q, bool walls, int state, int collision, const Launch& l, const PhaseArgs<T>& a);
// Fused hydrodynamic LB step (one launch).
template <typename T> cudaError_t launch_hydro(int Q, bool walls, int state, const Launch& l, const HydroArgs<T>& a);

// The same two kernels with two x-adjacent cells per thread (pair.cuh): l.block.x threads cover 2 l.block.x cells
// of a row; needs nx even.
template <typename T> cudaError_t launch_phase2(int Q, bool walls, int state, int collision, const Launch& l, const PhaseArgs<T>& a);
template <typename T> cudaError_t launch_hydro2(int Q, bool walls, int state, const Launch& l, const HydroArgs<T>& a);

// Algorithm 1, three launches each: stream h -> update phi -> collide h, and
// stream g -> update u (Uold -> Unew) -> collide g.  Two-grid storage only (a.Hsrc/a.Gsrc in ST_POST).
template <typename T> cudaError_t launch_unfused_phase(int Q, bool walls, int collision, const Launch& l, const PhaseArgs<T>& a);
template <typename T> cudaError_t launch_unfused_hydro(int Q, bool walls, const Launch& l, const HydroArgs<T>& a, const T* Uold, T* Unew);

// The two fused kernels in moment representation (ACM_OPT_MOMENTS; moment_impl.cuh), their initialiser and exports.
// local: the coefficient array of g holds the cell's own incoming populations (state right after acm_init).
template <typename T> cudaError_t launch_phase_mom(int Q, bool walls, const Launch& l, const MomPhaseArgs<T>& a);
template <typename T> cudaError_t launch_hydro_mom(int Q, bool walls, bool local, const Launch& l, const MomHydroArgs<T>& a);
// ... and as marching kernels: 32 x 8 tiles of columns marching along z over `zchunk` planes per block, the coefficient planes
// staged in shared memory by cp.async (the geometry's launch range [lz0, lz1) is split into chunks; l.grid / l.block are unused)
template <typename T> cudaError_t launch_phase_mom_march(int Q, bool walls, int zchunk, cudaStream_t stream, const MomPhaseArgs<T>& a);
template <typename T> cudaError_t launch_hydro_mom_march(int Q, bool walls, int zchunk, cudaStream_t stream, const MomHydroArgs<T>& a);
template <typename T> cudaError_t launch_init_mom(const Launch& l, const T* phi, const T* u, T* M, T* K, T* C, T* U0, T* U1, Geom g, size_t N);
template <typename T> cudaError_t launch_export_h_mom(int Q, const Launch& l, const T* M, const T* C, const T* Uo, T* out, Geom g, size_t N);
template <typename T>
cudaError_t launch_export_g_mom(int Q, bool local, const Launch& l, const T* K, const T* C, T* out, T* p, Geom g, size_t N, T rho_L, T drho);

// Equilibrium initialiser.
template <typename T>
cudaError_t launch_init(int Qh, int Qg, bool inplace, const Launch& l, const T* phi, const T* u, T* H, T* G, T* C, T* U, Geom g, size_t N, T ref);
// Export of a population array stored in `state` in the POST (post-collision at own cell) or
// incoming convention; optionally the pressure p = c_s^2 rho(phi) sum_i f_i.
template <typename T>
cudaError_t launch_export(int Q, int state, bool post, const Launch& l, const T* F, const T* C, T* out, T* p, Geom g, size_t N, T rho_L, T drho, T shift);
// Import: POST convention -> ST_SWAP storage, or incoming convention -> ST_POST storage.
template <typename T> cudaError_t launch_import(int Q, bool post, const Launch& l, const T* in, T* F, Geom g, size_t N, T shift);
// fp32 deviation storage (A22): out_i = in_i + shift w_i on the owned cells; out = in + shift on a whole field.
template <typename T> cudaError_t launch_shift_pop(int Q, const Launch& l, const T* in, T* out, Geom g, size_t N, T shift);
template <typename T> cudaError_t launch_shift_field(cudaStream_t s, const T* in, T* out, size_t n, T shift);

// Deterministic two-pass reductions.  `part` holds RED_BLOCKS * width partial sums followed by
// `width` results.
constexpr int RED_BLOCKS = 592, RED_THREADS = 256;   // 4 CTAs per SM on 148 SMs
constexpr int DIAG_WIDTH = 7;                        // V, V*x, V*y, V*z, V*ux, V*uy, V*uz
template <typename T> cudaError_t launch_sum_phi(cudaStream_t s, const T* C, size_t N, double* part);
// launch_bubble_diag sums over the owned planes [g.zlo, g.zhi); zshift = global z of plane 0 (slabs).
template <typename T> cudaError_t launch_bubble_diag(cudaStream_t s, const T* C, const T* U, Geom g, size_t N, int zshift, double ref, double* part);

}  // namespace acm
