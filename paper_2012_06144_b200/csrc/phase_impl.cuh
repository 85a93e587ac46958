// phase_impl.cuh -- fused phase-field LB kernel and its launcher, instantiated for one element
// type per translation unit (phase_f64.cu, phase_f32.cu define ACM_T and include this file).
#include "kernels.h"

namespace acm {

// ------------------------------------------------------------------------------------------
// Kernel 1: fused phase-field LB step (Alg. 2; eqs. 4-7, 23)
//   pull h -> phi_new = sum h -> grad/normal/theta from the OLD phi -> closed-form MRT collision
//   (first-order moments relaxed with omega_phi, all others with 1) -> store h, phi_new.
// With d = j - phi_new u + (theta/6) n:   h*_i = h^eq_i + F_i/2 + (1-omega_phi) 3 w_i e_i.d
// ------------------------------------------------------------------------------------------
template <typename T, int Q, bool WALLS, int STATE, int COLL>
__global__ void __launch_bounds__(ACM_MAXT, ACM_PHASE_MINB) phase_kernel(const PhaseArgs<T> a)
{
    int x, y, z;
    if (!cell_of_thread(a.g, x, y, z)) return;
    Nbr nb;
    nb.setup<WALLS>(a.g, x, y, z);
    const int idx = nb.at<0, 0, 0>();
    const size_t N = a.N;

    T h[Q];
    load_incoming<Q, T, WALLS, STATE>(a.Hsrc, N, nb, h);
    const T ux = __ldg(a.U + idx), uy = __ldg(a.U + N + idx), uz = __ldg(a.U + 2 * N + idx);
    const T c0 = __ldg(a.Csrc + idx);
    T gx, gy, gz, lap_unused;
    fd_phi<Q, T, false>(a.Csrc, nb, c0, gx, gy, gz, lap_unused);

    Moments<Q, T, false> m;
    m.compute(h);
    const T phi = m.m0;

    // interface normal (n = 0 where grad phi vanishes exactly) and theta = (1 - 4 (phi-1/2)^2)/xi
    const T g2 = gx * gx + gy * gy + gz * gz;
    const T inv = (g2 > T(0)) ? T(1) / sqrt(g2) : T(0);
    const T dc = c0 - T(0.5);
    const T theta = (T(1) - T(4) * dc * dc) * a.inv_xi;
    const T tnx = theta * inv * gx, tny = theta * inv * gy, tnz = theta * inv * gz;   // theta * n

    // closed form of the collision: h*_i = w_i [A + e_i.b + e_i e_i : T] (+ keep * h_i for SRT)
    T A, bx, by, bz, Ts, keep;
    if constexpr (COLL == PHASE_MRT) {
        // first-order moments relaxed with omega_phi, all others with 1 (A3):
        // with d = j - phi u + (theta/6) n:  h*_i = phi Gamma_i(u) + F_i/2 + (1-omega) 3 w_i e_i.d
        const T k = T(3) * a.one_minus_omega;
        const T sixth = T(1.0 / 6.0);
        const T dxm = m.jx - phi * ux + sixth * tnx;
        const T dym = m.jy - phi * uy + sixth * tny;
        const T dzm = m.jz - phi * uz + sixth * tnz;
        const T p3 = T(3) * phi;
        A = phi * (T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz));
        bx = p3 * ux + T(0.5) * tnx + k * dxm;
        by = p3 * uy + T(0.5) * tny + k * dym;
        bz = p3 * uz + T(0.5) * tnz + k * dzm;
        Ts = T(4.5) * phi;
        keep = T(0);
    } else {
        // single relaxation time (A23): h*_i = (1-omega) h_i + omega phi Gamma_i(u) + (1-omega/2) F_i
        const T omega = T(1) - a.one_minus_omega;
        const T op = omega * phi, fh = T(1) - T(0.5) * omega;
        A = op * (T(1) - T(1.5) * (ux * ux + uy * uy + uz * uz));
        bx = T(3) * op * ux + fh * tnx;
        by = T(3) * op * uy + fh * tny;
        bz = T(3) * op * uz + fh * tnz;
        Ts = T(4.5) * op;
        keep = a.one_minus_omega;
    }
    auto post = [&](auto ic, T v) -> T {
        if constexpr (COLL == PHASE_SRT) return v + keep * h[decltype(ic)::value];
        else return v;
    };
    if constexpr (sizeof(T) == 8) {
        emit_populations<Q, T>(A, bx, by, bz, Ts * ux * ux, Ts * uy * uy, Ts * uz * uz, Ts * ux * uy, Ts * ux * uz,
                               Ts * uy * uz, [&](auto ic, T v) {
                                   st_stream(outgoing_ptr<Q, decltype(ic)::value, T, WALLS, STATE>(a.Hdst, N, nb), post(ic, v));
                               });
    } else {
        // fp32 instance (reading A22): the rest population is set by subtraction,
        // h*_0 = phi_new - sum_{i>=1} h*_i, so that the collision conserves phi exactly in fp32.
        T rest = phi;
        emit_populations<Q, T>(A, bx, by, bz, Ts * ux * ux, Ts * uy * uy, Ts * uz * uz, Ts * ux * uy, Ts * ux * uz,
                               Ts * uy * uz, [&](auto ic, T v) {
                                   constexpr int i = decltype(ic)::value;
                                   if constexpr (i > 0) {
                                       const T o = post(ic, v);
                                       rest -= o;
                                       st_stream(outgoing_ptr<Q, i, T, WALLS, STATE>(a.Hdst, N, nb), o);
                                   }
                               });
        st_stream(outgoing_ptr<Q, 0, T, WALLS, STATE>(a.Hdst, N, nb), rest);
    }
    a.Cdst[idx] = phi;
}

template <typename T, int Q, bool WALLS, int STATE>
static void launch_phase_coll(int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (collision == PHASE_SRT) phase_kernel<T, Q, WALLS, STATE, PHASE_SRT><<<l.grid, l.block, 0, l.stream>>>(a);
    else phase_kernel<T, Q, WALLS, STATE, PHASE_MRT><<<l.grid, l.block, 0, l.stream>>>(a);
}

template <typename T, int Q, bool WALLS>
static void launch_phase_state(int state, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (state == ST_POST) launch_phase_coll<T, Q, WALLS, ST_POST>(collision, l, a);
    else if (state == ST_IN) launch_phase_coll<T, Q, WALLS, ST_IN>(collision, l, a);
    else launch_phase_coll<T, Q, WALLS, ST_SWAP>(collision, l, a);
}

template <typename T, int Q>
static void launch_phase_q(bool walls, int state, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (walls) launch_phase_state<T, Q, true>(state, collision, l, a);
    else launch_phase_state<T, Q, false>(state, collision, l, a);
}

template <typename T>
cudaError_t launch_phase(int Q, bool walls, int state, int collision, const Launch& l, const PhaseArgs<T>& a)
{
    if (Q == 15) launch_phase_q<T, 15>(walls, state, collision, l, a);
    else if (Q == 19) launch_phase_q<T, 19>(walls, state, collision, l, a);
    else launch_phase_q<T, 27>(walls, state, collision, l, a);
    return cudaGetLastError();
}

template cudaError_t launch_phase<ACM_T>(int, bool, int, int, const Launch&, const PhaseArgs<ACM_T>&);

}  // namespace acm
