// Fused annealing step for non-Boolean SAT ("W_mi has q > 2 states").
//
// Every variable has q states and q fields, P_i = softmax(h_i).  Energy Eq.8: a clause counts
// when no variable takes its clause value W_mi; mean field U = sum_m prod_{i in dm} [1 - P_i(W_mi)] (Eq.11);
//   dU/dP_i(s) = - sum_{m ni i, W_mi = s} prod_{k in dm, k != i} [1 - P_k(W_mk)]                    (S28)
//   g^p_i(s) = dU/dP_i(s) + (1/beta)[ln P_i(s) + 1],   g^h_i(s) = gamma P_i(s)[g^p_i(s) - sum_s' P_i(s') g^p_i(s')]   (S20)
// followed by the optimiser update, all in registers: rows a1-a4 of DESIGN.md section 2 in one launch.
//
// Layout: the Potts one, field (i, s, r) of a replica block at (i*q + s)*Rb + r.  One thread owns VEC consecutive replicas
// of ALL q states of one variable (q <= 8): the sums over states are register adds.  The gathered quantity is the centred
// marginal D = P - 1/q as in the Potts kernels (1 - P = (1 - 1/q) - D).  The occurrence table is keyed by (variable, clause
// value): row i*q + s lists the clauses that hold variable i with W_mi = s, each as the gather ROWS k*q + W_mk of its other
// variables (stride padded to a power of two; pad entries name row n*q and contribute the factor 1), in clause order,
// which is the oracle's summation order.  No atomics (north_star subsystem 3, per state).
//
// The paper gives this variant one sentence and no workload; the kernel is written for correctness and parity (thread per
// variable, occurrence lists walked serially), not tuned: DESIGN.md section 13.
#include "device_math.cuh"

namespace fem {

template <typename T>
struct QsatParams {
    BlockArrays<T> a;
    DevProblem dp;
    Sc<T> sc;
    T *g_other;      // prepare mode: the other gather buffer (its pad row is cleared too)
    unsigned rv;     // Rb / VEC lanes per variable
    unsigned total;  // n * rv threads per replica block
};

constexpr int kQsatMaxQ = 8;

template <typename T, int VEC, bool STEP>
__global__ void __launch_bounds__(kThreads) qsat_kernel(const QsatParams<T> p) {
    using R = Row<T, VEC>;
    pdl_trigger();
    const unsigned idx = blockIdx.x * kThreads + threadIdx.x;
    if (idx >= p.total) return;
    const unsigned i = idx / p.rv;
    const unsigned c = (idx - i * p.rv) * VEC;
    const int q = p.dp.q, n = p.dp.n;
    const unsigned Rb = p.a.Rb;
    const int64_t blk = (int64_t)blockIdx.y * p.a.blk_stride;
    const int64_t off0 = blk + ((int64_t)i * q * Rb + c);  // state s: + s * Rb
    const T *__restrict__ gin = p.a.g_in + blk + c;
    const Sc<T> &sc = p.sc;
    const T inv_q = (T)1 / (T)q;
    const T one_minus = (T)1 - inv_q;
    const unsigned pad_row = (unsigned)n * (unsigned)q;
    const int kst = p.dp.kstride <= 1 ? 1 : (p.dp.kstride <= 2 ? 2 : (p.dp.kstride <= 4 ? 4 : 8));  // entries per occurrence

    pdl_wait();  // everything below reads or overwrites what the previous launch wrote
    T h[kQsatMaxQ][VEC];
#pragma unroll
    for (int s = 0; s < kQsatMaxQ; ++s) {
        if (s < q) {
            const R r = R::ld_stream(p.a.h + off0 + (int64_t)s * Rb);
#pragma unroll
            for (int v = 0; v < VEC; ++v) h[s][v] = r.v[v];
        } else {
#pragma unroll
            for (int v = 0; v < VEC; ++v) h[s][v] = (T)-3.0e38;
        }
    }
    if (STEP) {
        // ---- dU/dP_i(s) = -f(s): leave-one-out products of the clauses that hold (i, s), by multiplication only
        T gp[kQsatMaxQ][VEC];
#pragma unroll
        for (int s = 0; s < kQsatMaxQ; ++s) {
#pragma unroll
            for (int v = 0; v < VEC; ++v) gp[s][v] = (T)0;
            if (s < q) {
                const int o0 = __ldg(p.dp.occ_ptr + i * q + s), o1 = __ldg(p.dp.occ_ptr + i * q + s + 1);
                T f[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) f[v] = (T)0;
                for (int o = o0; o < o1; ++o) {
                    T prod[VEC];
#pragma unroll
                    for (int v = 0; v < VEC; ++v) prod[v] = (T)1;
                    for (int x = 0; x < kst; ++x) {
                        const unsigned row = (unsigned)__ldg(p.dp.occ + (int64_t)o * kst + x);
                        const R nb = R::ld(gin + (unsigned long long)row * Rb);
#pragma unroll
                        for (int v = 0; v < VEC; ++v) prod[v] *= row == pad_row ? (T)1 : one_minus - nb.v[v];
                    }
#pragma unroll
                    for (int v = 0; v < VEC; ++v) f[v] += prod[v];
                }
#pragma unroll
                for (int v = 0; v < VEC; ++v) gp[s][v] = fma(h[s][v], sc.inv_beta, -f[v]);  // (the "+1" of S26 cancels in S20)
            }
        }
        // ---- softmax, <g^p>_P, chain rule and optimiser, state by state for the moments
        T P[kQsatMaxQ][VEC], gbar[VEC];
#pragma unroll
        for (int v = 0; v < VEC; ++v) {
            T mx = h[0][v];
#pragma unroll
            for (int s = 1; s < kQsatMaxQ; ++s) mx = fmax(mx, h[s][v]);
            T z = (T)0;
#pragma unroll
            for (int s = 0; s < kQsatMaxQ; ++s) {
                P[s][v] = s < q ? fexp(h[s][v] - mx) : (T)0;
                z += P[s][v];
            }
            const T rz = frcp(z);
            gbar[v] = (T)0;
#pragma unroll
            for (int s = 0; s < kQsatMaxQ; ++s) {
                P[s][v] *= rz;
                gbar[v] = fma(P[s][v], gp[s][v], gbar[v]);
            }
        }
        const bool use_m1 = sc.uses_m1(), use_m2 = sc.uses_m2();
#pragma unroll
        for (int s = 0; s < kQsatMaxQ; ++s) {
            if (s < q) {
                const int64_t off = off0 + (int64_t)s * Rb;
                R m1 = {}, m2 = {}, hn;
                if (use_m1) m1 = R::ld_stream(p.a.m1 + off);
                if (use_m2) m2 = R::ld_stream(p.a.m2 + off);
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const T g = sc.gamma * (P[s][v] * (gp[s][v] - gbar[v]));
                    hn.v[v] = opt_update(h[s][v], g, m1.v[v], m2.v[v], sc);
                    h[s][v] = hn.v[v];
                }
                hn.st_stream(p.a.h + off);
                if (use_m1) m1.st_stream(p.a.m1 + off);
                if (use_m2) m2.st_stream(p.a.m2 + off);
            }
        }
    }
    // ---- centred marginals of the (new) fields -> the gather buffer of the next step
#pragma unroll
    for (int v = 0; v < VEC; ++v) {
        T mx = h[0][v];
#pragma unroll
        for (int s = 1; s < kQsatMaxQ; ++s) mx = fmax(mx, h[s][v]);
        T z = (T)0;
#pragma unroll
        for (int s = 0; s < kQsatMaxQ; ++s) {
            h[s][v] = s < q ? fexp(h[s][v] - mx) : (T)0;
            z += h[s][v];
        }
        const T rz = frcp(z);
#pragma unroll
        for (int s = 0; s < kQsatMaxQ; ++s) h[s][v] = fma(h[s][v], rz, -inv_q);
    }
#pragma unroll
    for (int s = 0; s < kQsatMaxQ; ++s) {
        if (s < q) {
            R po;
#pragma unroll
            for (int v = 0; v < VEC; ++v) po.v[v] = h[s][v];
            po.st(p.a.g_out + off0 + (int64_t)s * Rb);
        }
    }
    if (!STEP && i == 0) {  // the pad row of both gather buffers (never used as a factor, but it is read)
        R zero;
#pragma unroll
        for (int v = 0; v < VEC; ++v) zero.v[v] = (T)0;
        zero.st(p.a.g_out + blk + ((int64_t)pad_row * Rb + c));
        zero.st(p.g_other + blk + ((int64_t)pad_row * Rb + c));
    }
}

template <typename T>
static void launch_qsat_t(Handle *hd, const StepScalars &sc, bool step, int blk_begin, int blk_count) {
    using S = StateOf<T>;
    const int Rb = hd->Rb;
    const int64_t base = (int64_t)blk_begin * hd->rows * Rb;
    QsatParams<T> p;
    p.a.h = S::h(hd) + base;
    p.a.m1 = S::m1(hd) + base;
    p.a.m2 = S::m2(hd) + base;
    p.a.g_in = S::g(hd, hd->cur) + base;
    p.a.g_out = (step ? S::g(hd, hd->cur ^ 1) : S::g(hd, hd->cur)) + base;
    p.g_other = S::g(hd, hd->cur ^ 1) + base;
    p.a.blk_stride = hd->rows * Rb;
    p.a.Rb = Rb;
    p.dp = hd->dp;
    p.sc = Sc<T>(sc);
    const int VEC = (Rb % 4 == 0) ? 4 : 1;
    p.rv = (unsigned)(Rb / VEC);
    p.total = (unsigned)hd->dp.n * p.rv;
    dim3 grid((unsigned)ceil_div(p.total, kThreads), (unsigned)blk_count);
    if (VEC == 4) {
        if (step) launch_pdl(qsat_kernel<T, 4, true>, grid, dim3(kThreads), hd->stream, p);
        else launch_pdl(qsat_kernel<T, 4, false>, grid, dim3(kThreads), hd->stream, p);
    } else {
        if (step) launch_pdl(qsat_kernel<T, 1, true>, grid, dim3(kThreads), hd->stream, p);
        else launch_pdl(qsat_kernel<T, 1, false>, grid, dim3(kThreads), hd->stream, p);
    }
    hd->launches++;
}

// step == false: centred marginals of the current fields into g[cur] (and the pad rows of both gather buffers)
void launch_qsat(Handle *hd, const StepScalars &sc, bool wide, bool step, int blk_begin, int blk_count) {
    if (wide) launch_qsat_t<double>(hd, sc, step, blk_begin, blk_count);
    else launch_qsat_t<float>(hd, sc, step, blk_begin, blk_count);
}

}  // namespace fem
