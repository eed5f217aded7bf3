// Device helpers shared by the step kernels: vector row access and the two-state / Adam arithmetic.
#pragma once
#include <type_traits>

#include "fem_internal.cuh"

namespace fem {

// ---- VEC-wide row access (VEC = 1, 2 or 4 consecutive replicas) of storage type T ----
// T = float: the bulk of the anneal.  T = double: the "wide" phase (first precise_steps steps), where
// both the arithmetic and the stored state are fp64.
template <typename T, int VEC>
struct Row {
    T v[VEC];
    // 16-byte vector type that carries the row
    using V16 = typename std::conditional<sizeof(T) == 4, float4, double2>::type;
    static constexpr int kPer16 = 16 / sizeof(T);
    static constexpr int kBytes = VEC * sizeof(T);

    __device__ __forceinline__ static Row ld(const T *p) {  // read-only path (gathers)
        Row r;
        if constexpr (kBytes >= 16) {
#pragma unroll
            for (int k = 0; k < kBytes / 16; ++k) {
                const V16 t = __ldg(reinterpret_cast<const V16 *>(p) + k);
                memcpy(&r.v[k * kPer16], &t, 16);
            }
        } else if constexpr (kBytes == 8) {
            const float2 t = __ldg(reinterpret_cast<const float2 *>(p));
            memcpy(&r.v[0], &t, 8);
        } else {
            r.v[0] = __ldg(p);
        }
        return r;
    }
    __device__ __forceinline__ static Row ld_stream(const T *p) {  // streamed once: evict-first
        Row r;
        if constexpr (kBytes >= 16) {
#pragma unroll
            for (int k = 0; k < kBytes / 16; ++k) {
                const V16 t = __ldcs(reinterpret_cast<const V16 *>(p) + k);
                memcpy(&r.v[k * kPer16], &t, 16);
            }
        } else if constexpr (kBytes == 8) {
            const float2 t = __ldcs(reinterpret_cast<const float2 *>(p));
            memcpy(&r.v[0], &t, 8);
        } else {
            r.v[0] = __ldcs(p);
        }
        return r;
    }
    __device__ __forceinline__ void st(T *p) const {
        if constexpr (kBytes >= 16) {
#pragma unroll
            for (int k = 0; k < kBytes / 16; ++k) {
                V16 t;
                memcpy(&t, &v[k * kPer16], 16);
                reinterpret_cast<V16 *>(p)[k] = t;
            }
        } else if constexpr (kBytes == 8) {
            float2 t;
            memcpy(&t, &v[0], 8);
            *reinterpret_cast<float2 *>(p) = t;
        } else {
            *p = v[0];
        }
    }
    __device__ __forceinline__ void st_stream(T *p) const {
        if constexpr (kBytes >= 16) {
#pragma unroll
            for (int k = 0; k < kBytes / 16; ++k) {
                V16 t;
                memcpy(&t, &v[k * kPer16], 16);
                __stcs(reinterpret_cast<V16 *>(p) + k, t);
            }
        } else if constexpr (kBytes == 8) {
            float2 t;
            memcpy(&t, &v[0], 8);
            __stcs(reinterpret_cast<float2 *>(p), t);
        } else {
            __stcs(p, v[0]);
        }
    }
};

// ---- compact gather buffer of the manipulated gradients ----
// With one-hot neighbours (S25/S27/S30) the gathered quantity is an integer: sgn(m_j) in {-1, 0, +1} for the
// two-state kinds, the state id argmax_s h_j(s) for the Potts kind.  It is stored as ONE BYTE per (variable,
// replica) -- element (i, r) of a replica block at byte i*Rb + r of the fp32 gather array's memory -- so a
// neighbour gather moves 1 byte where the exact gradient moves 4 (two-state) or 4q (Potts) bytes
// (SURVEY.md section 8(f) row 1).  VEC consecutive replicas travel as one 8-, 16- or 32-bit access.
template <int VEC>
__device__ __forceinline__ void ld_bytes(const signed char *p, int (&out)[VEC]) {
    if constexpr (VEC == 4) {
        const int w = __ldg(reinterpret_cast<const int *>(p));
#pragma unroll
        for (int v = 0; v < 4; ++v) out[v] = (int)(signed char)((w >> (8 * v)) & 0xff);
    } else if constexpr (VEC == 2) {
        const short w = __ldg(reinterpret_cast<const short *>(p));
        out[0] = (int)(signed char)(w & 0xff);
        out[1] = (int)(signed char)((w >> 8) & 0xff);
    } else {
        out[0] = (int)__ldg(p);
    }
}
// the same VEC bytes left packed in one word (byte v = replica v), for kernels that keep many neighbours in flight
template <int VEC>
__device__ __forceinline__ unsigned ld_bytes_packed(const signed char *p) {
    if constexpr (VEC == 4) return (unsigned)__ldg(reinterpret_cast<const int *>(p));
    else if constexpr (VEC == 2) return (unsigned)(unsigned short)__ldg(reinterpret_cast<const short *>(p));
    else return (unsigned)(unsigned char)__ldg(p);
}
template <int VEC>
__device__ __forceinline__ void st_bytes(signed char *p, const int (&in)[VEC]) {
    if constexpr (VEC == 4) {
        *reinterpret_cast<int *>(p) = (in[0] & 0xff) | ((in[1] & 0xff) << 8) | ((in[2] & 0xff) << 16) | ((in[3] & 0xff) << 24);
    } else if constexpr (VEC == 2) {
        *reinterpret_cast<short *>(p) = (short)((in[0] & 0xff) | ((in[1] & 0xff) << 8));
    } else {
        *p = (signed char)in[0];
    }
}

// ---- programmatic dependent launch (PDL): consecutive step kernels overlap launch latency and tail ----
// pdl_trigger lets the NEXT kernel in the stream start being scheduled once every CTA of this grid has
// started; pdl_wait blocks until the PREVIOUS grid has completed and its writes are visible.  Only loads
// of the static problem structure may precede pdl_wait.
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t stream, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = 0;
    cfg.stream = stream;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, args...);
}

// ---- per-step scalars in the compute type (narrowed once on the host, not per thread) ----
// opt = 0 Adam: b1, b2, omb1 = 1-b1, omb2 = 1-b2, step_size = lr/(1-b1^t), rsqrt_bc2 = 1/sqrt(1-b2^t)
// opt = 1 RMSprop: b1 = momentum, b2 = alpha, omb2 = 1-alpha, step_size = lr
// opt = 2 SGD: b1 = momentum, omb1 = 1-dampening, step_size = lr, first = 1 at the first step of the anneal
template <typename T>
struct Sc {
    T inv_beta, step_size, rsqrt_bc2, eps, b1, b2, omb1, omb2, wd, two_lambda;
    T gamma;    // gamma_grad of S20; 1 for the exact gradient
    int opt;    // 0 Adam, 1 RMSprop, 2 SGD
    int first;  // SGD: the momentum buffer starts as the first gradient
    int disc;   // manipulated gradients (S25/S27/S30): neighbours enter as one-hot vectors, coupling term normalised
    Sc() = default;
    __host__ explicit Sc(const StepScalars &s)
        : inv_beta((T)s.inv_beta), step_size((T)s.step_size), rsqrt_bc2((T)s.rsqrt_bc2), eps((T)s.eps), b1((T)s.b1),
          b2((T)s.b2), omb1((T)s.one_minus_b1), omb2((T)s.one_minus_b2), wd((T)s.wd), two_lambda((T)s.two_lambda),
          gamma((T)s.gamma), opt(s.opt), first(s.first), disc(s.disc) {}
    // which moment arrays the optimiser touches (the others are neither read nor written: 8 B per field each)
    __host__ __device__ bool uses_m1() const { return opt == 0 || b1 > (T)0; }
    __host__ __device__ bool uses_m2() const { return opt != 2; }
};

// fp64 (wide phase): accurate libm.  fp32 (bulk): hardware approximations (ex2/rcp/sqrt MUFU ops, <= 2 ulp),
// which sit at the level of the fp32 storage rounding of the state itself.
__device__ __forceinline__ double fexp(double x) { return exp(x); }
__device__ __forceinline__ float fexp(float x) {  // exp via ex2.approx; results below 2^-126 flush to 0 (harmless here)
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x * 1.4426950408889634f));
    return y;
}
__device__ __forceinline__ double fsqrt(double x) { return sqrt(x); }
__device__ __forceinline__ float fsqrt(float x) {
    float y;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ double flog(double x) { return log(x); }
__device__ __forceinline__ float flog(float x) { return __logf(x); }
__device__ __forceinline__ double fdiv(double a, double b) { return a / b; }
__device__ __forceinline__ float fdiv(float a, float b) {
    float y;
    asm("div.approx.ftz.f32 %0, %1, %2;" : "=f"(y) : "f"(a), "f"(b));
    return y;
}
__device__ __forceinline__ double frcp(double x) { return 1.0 / x; }
__device__ __forceinline__ float frcp(float x) {
    float y;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

// Two-state pieces from one field h = h(+1) - h(-1):
//   p(1-p) = e/(1+e)^2 with e = exp(-|h|)   (exact in the saturated tails, where 1 - m^2 would round to 0)
//   m = 2p - 1 = tanh(h/2)
// fp64: library tanh keeps RELATIVE accuracy for |h| -> 0, where the deviation from the uniform marginal is all
// the signal there is (the start of the anneal, which the wide phase covers).  fp32: m = sign(h)(1-e)/(1+e),
// absolute accuracy ~6e-8, one exp shared with nothing else to compute.
template <typename T>
__device__ __forceinline__ T p1mp_of(T h) {
    const T e = fexp(-fabs(h));
    const T r = frcp((T)1 + e);
    return e * r * r;
}
__device__ __forceinline__ double mag_of(double h) { return tanh(0.5 * h); }
__device__ __forceinline__ float mag_of(float h) {
    const float e = fexp(-fabsf(h));
    const float am = (1.0f - e) * frcp(1.0f + e);
    return copysignf(am, h);
}
template <typename T>
__device__ __forceinline__ T sigmoid_of(T h) {
    const T e = fexp(-fabs(h));
    const T r = frcp((T)1 + e);
    return h < (T)0 ? e * r : r;
}

// Optimiser update (Adam, RMSprop and SGD "as provided by PyTorch"): returns the new field.
//   Adam    : Kingma & Ba as arranged by torch.optim.Adam
//   RMSprop : v = alpha v + (1-alpha) g^2; d = g / (sqrt(v) + eps); momentum: b = mom b + d, h -= lr b; else h -= lr d
//   SGD     : b = g at the first step, b = mom b + (1-dampening) g after; h -= lr b   (mom = 0: h -= lr g)
// m1 is Adam's first moment / the momentum buffer b, m2 is Adam's second moment / RMSprop's v.
// Every multiply-add is written as an explicit fma so that all kernels (stepwise, persistent, Potts, dense) round
// alike whatever contraction the compiler would have picked.
template <typename T>
__device__ __forceinline__ T opt_update(T h, T g, T &m1, T &m2, const Sc<T> &sc) {
    g = fma(sc.wd, h, g);
    if (sc.opt == 0) {
        m1 = fma(sc.b1, m1, sc.omb1 * g);
        m2 = fma(sc.b2, m2, (sc.omb2 * g) * g);
        const T denom = fma(fsqrt(m2), sc.rsqrt_bc2, sc.eps);
        return fma(-sc.step_size, fdiv(m1, denom), h);
    }
    if (sc.opt == 1) {
        m2 = fma(sc.b2, m2, (sc.omb2 * g) * g);
        const T d = fdiv(g, fsqrt(m2) + sc.eps);
        if (sc.b1 > (T)0) {
            m1 = fma(sc.b1, m1, d);
            return fma(-sc.step_size, m1, h);
        }
        return fma(-sc.step_size, d, h);
    }
    if (sc.b1 > (T)0) {
        m1 = sc.first ? g : fma(sc.b1, m1, sc.omb1 * g);
        return fma(-sc.step_size, m1, h);
    }
    return fma(-sc.step_size, g, h);
}

// Two-state field gradient S29: g^h = gamma [c_i dU/dp + h/beta] p(1-p), ln(p/(1-p)) = h.  c_i = 1 and
// gamma = 1 give the exact gradient.  The fused multiply-add is written out so that every kernel rounds alike.
template <typename T>
__device__ __forceinline__ T q2_grad(T dU, T ci, T h, const Sc<T> &sc) {
    const T cd = ci * dU;
    return sc.gamma * (fma(h, sc.inv_beta, cd) * p1mp_of(h));
}

// sgn(m) = sgn(h) with sgn(0) = 0: the two-state one-hot vector as a magnetisation, 2 e(+1) - 1 (S29)
template <typename T>
__device__ __forceinline__ T sign_of(T h) {
    return h > (T)0 ? (T)1 : (h < (T)0 ? (T)-1 : (T)0);
}

}  // namespace fem
