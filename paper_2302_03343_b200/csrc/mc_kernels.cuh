// mc_kernels.cuh -- the Monte Carlo steps around the PDF hot path:
// RAMBO phase space (eq. 1.103-1.110; p_T cut L2070), the VEGAS importance-sampling step
// (eq. 1.74-1.75, 1.80-1.83, L866-935) and the unweighting rule (L2028-2030).  Pure fp64 ALU / streaming kernels:
// one thread per event, coalesced loads and stores, block-level reductions before the global atomics.
// Part of the CUDA product path; shares nothing with oracle/.
#pragma once
#include <cuda_runtime.h>

namespace pdfg {

constexpr int kRamboMaxN = 16;
struct RamboMasses { int massive; double m[kRamboMaxN]; };

// eq. 1.108 (the Gamma functions of small integers are factorials)
__host__ __device__ inline double rambo_w0(int n, double s)
{
    const double twopi = 6.283185307179586476925286766559, halfpi = 1.5707963267948966192313216916398;
    double f = 1.0;                                        // Gamma(n) Gamma(n-1) = (n-1)! (n-2)!
    for (int k = 2; k <= n - 1; ++k) f *= (double)k;
    double g = 1.0;
    for (int k = 2; k <= n - 2; ++k) g *= (double)k;
    return pow(twopi, 4.0 - 3.0 * n) * pow(halfpi, n - 1.0) * pow(s, n - 2.0) / (f * g);
}

// one thread per event.  Pass 1 builds Q = sum q_i (eq. 1.107), pass 2 regenerates every q_i from its uniforms
// (cheaper than keeping 4 n doubles per thread) and applies the boost and scaling of eq. 1.103-1.104.  The massive
// case rescales by xi (Newton's iteration on the energy constraint below eq. 1.109) and multiplies w_m (eq. 1.110).
__global__ void __launch_bounds__(128)
k_rambo(long long nev, int n, const double *__restrict__ sqrt_s, const __grid_constant__ RamboMasses mass,
        const double *__restrict__ u, double ptmin, double *__restrict__ p, double *__restrict__ w)
{
    const long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= nev) return;
    const double4 *ue = reinterpret_cast<const double4 *>(u) + e * n;
    double4 *pe = reinterpret_cast<double4 *>(p) + e * n;
    const double twopi = 6.283185307179586476925286766559;
    auto make_q = [&](int i) {
        const double2 r01 = __ldcs(reinterpret_cast<const double2 *>(ue + i)), r23 = __ldcs(reinterpret_cast<const double2 *>(ue + i) + 1);
        const double4 r = make_double4(r01.x, r01.y, r23.x, r23.y);
        const double c = 2.0 * r.x - 1.0, phi = twopi * r.y, q0 = -log(r.z * r.w), st = sqrt(1.0 - c * c);
        double sn, cs;
        sincos(phi, &sn, &cs);
        return make_double4(q0, q0 * st * cs, q0 * st * sn, q0 * c);
    };
    double Q0 = 0.0, Q1 = 0.0, Q2 = 0.0, Q3 = 0.0;
    for (int i = 0; i < n; ++i) { const double4 q = make_q(i); Q0 += q.x; Q1 += q.y; Q2 += q.z; Q3 += q.w; }
    const double rs = sqrt_s[e], s = rs * rs;
    if (mass.massive) {                                 // closed threshold (DESIGN R-6): no phase space, weight 0
        double sm = 0.0;
        for (int i = 0; i < n; ++i) sm += mass.m[i];
        if (!(rs > sm)) {
            for (int i = 0; i < n; ++i) pe[i] = make_double4(0.0, 0.0, 0.0, 0.0);
            w[e] = 0.0;
            return;
        }
    }
    const double M = sqrt(Q0 * Q0 - Q1 * Q1 - Q2 * Q2 - Q3 * Q3);
    const double b1 = -Q1 / M, b2 = -Q2 / M, b3 = -Q3 / M, gamma = Q0 / M, a = 1.0 / (1.0 + gamma), x = rs / M;
    double wt = rambo_w0(n, s);
    double E[kRamboMaxN];
    bool cut = false;
    for (int i = 0; i < n; ++i) {
        const double4 q = make_q(i);
        const double bq = b1 * q.y + b2 * q.z + b3 * q.w;
        double4 k;
        k.x = x * (gamma * q.x + bq);
        k.y = x * (q.y + b1 * q.x + a * bq * b1);
        k.z = x * (q.z + b2 * q.x + a * bq * b2);
        k.w = x * (q.w + b3 * q.x + a * bq * b3);
        E[i] = k.x;
        if (!mass.massive) {
            cut |= sqrt(k.y * k.y + k.z * k.z) < ptmin;
            pe[i] = k;
        }
    }
    if (mass.massive) {
        double sm = 0.0;
        for (int i = 0; i < n; ++i) sm += mass.m[i];
        double xi = sqrt(1.0 - (sm / rs) * (sm / rs));
        for (int it = 0; it < 100; ++it) {
            double g = -rs, dg = 0.0;
            for (int i = 0; i < n; ++i) {
                const double k0 = sqrt(mass.m[i] * mass.m[i] + xi * xi * E[i] * E[i]);
                g += k0;
                dg += xi * E[i] * E[i] / k0;
            }
            const double step = g / dg;
            xi -= step;
            if (fabs(step) <= 1e-15 * xi) break;
        }
        double sk = 0.0, prod = 1.0, sk2 = 0.0;
        for (int i = 0; i < n; ++i) {
            const double4 q = make_q(i);
            const double bq = b1 * q.y + b2 * q.z + b3 * q.w;
            const double kabs = xi * E[i], k0 = sqrt(mass.m[i] * mass.m[i] + kabs * kabs);
            double4 k;
            k.x = k0;
            k.y = xi * (x * (q.y + b1 * q.x + a * bq * b1));
            k.z = xi * (x * (q.z + b2 * q.x + a * bq * b2));
            k.w = xi * (x * (q.w + b3 * q.x + a * bq * b3));
            cut |= sqrt(k.y * k.y + k.z * k.z) < ptmin;
            pe[i] = k;
            sk += kabs; prod *= kabs / k0; sk2 += kabs * kabs / k0;
        }
        wt *= pow(s, 2.0 - n) * pow(sk, 2.0 * n - 3.0) * prod / sk2;
    }
    w[e] = (ptmin > 0.0 && cut) ? 0.0 : wt;
}

// ---- VEGAS ---------------------------------------------------------------------------------------
// eq. 1.81: uniforms through the per-dimension bin edges (staged in shared memory); one thread per point
__global__ void __launch_bounds__(256)
k_vegas_map(int ndim, int nb, const double *__restrict__ edges, long long n, const double *__restrict__ u,
            double *__restrict__ x, double *__restrict__ jac, int *__restrict__ bin)
{
    extern __shared__ double s_ve[];
    double *s_e = s_ve;
    for (int k = threadIdx.x; k < ndim * (nb + 1); k += blockDim.x) s_e[k] = edges[k];
    __syncthreads();
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        double j = 1.0;
        for (int d = 0; d < ndim; ++d) {
            const double y = u[e * ndim + d] * nb;
            int k = (int)y;
            k = k > nb - 1 ? nb - 1 : (k < 0 ? 0 : k);
            const double lo = s_e[d * (nb + 1) + k], width = s_e[d * (nb + 1) + k + 1] - lo;
            x[e * ndim + d] = lo + (y - k) * width;
            j *= nb * width;
            if (bin) bin[e * ndim + d] = k;
        }
        jac[e] = j;
    }
}

// eq. 1.74-1.75 sums and the per-bin |f/p| histograms (L913): per-CTA partial sums in shared memory (warp shuffles
// for the two scalars, shared-memory atomics for the bins), then one global atomic per CTA and value
__global__ void __launch_bounds__(256)
k_vegas_accumulate(int ndim, int nb, long long n, const double *__restrict__ f, const double *__restrict__ jac,
                   const int *__restrict__ bin, double *__restrict__ sums, double *__restrict__ hist)
{
    extern __shared__ double s_vh[];                       // [ndim * nb] + [2 * 8]
    double *s_h = s_vh, *s_part = s_h + ndim * nb;
    for (int k = threadIdx.x; k < ndim * nb + 16; k += blockDim.x) s_h[k] = 0.0;
    __syncthreads();
    double a = 0.0, b = 0.0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const double fw = f[e] * jac[e];
        a += fw; b += fw * fw;
        if (hist) for (int d = 0; d < ndim; ++d) atomicAdd(s_h + d * nb + bin[e * ndim + d], fabs(fw));
    }
    for (int o = 16; o; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); b += __shfl_xor_sync(0xffffffffu, b, o); }
    if ((threadIdx.x & 31) == 0) { s_part[2 * (threadIdx.x >> 5)] = a; s_part[2 * (threadIdx.x >> 5) + 1] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sa = 0.0, sb = 0.0;
        for (int k = 0; k < (int)(blockDim.x >> 5); ++k) { sa += s_part[2 * k]; sb += s_part[2 * k + 1]; }
        atomicAdd(sums, sa); atomicAdd(sums + 1, sb);
    }
    if (hist) for (int k = threadIdx.x; k < ndim * nb; k += blockDim.x) if (s_h[k] != 0.0) atomicAdd(hist + k, s_h[k]);
}

// grid refinement: one CTA, one thread per dimension walks the cumulative (damped) histogram and cuts it in nb
// equal shares, linear inside an old bin (L913; alpha = 1: no damping)
__global__ void k_vegas_refine(int ndim, int nb, const double *__restrict__ hist, double alpha, double *__restrict__ edges,
                               double *__restrict__ scratch /*[ndim][2 nb + 1]*/)
{
    const int d = blockIdx.x * blockDim.x + threadIdx.x;
    if (d >= ndim) return;
    double *ed = edges + (size_t)d * (nb + 1);
    double *h = scratch + (size_t)d * (2 * nb + 1), *ne = h + nb;
    double tot = 0.0;
    for (int k = 0; k < nb; ++k) tot += hist[d * nb + k];
    if (!(tot > 0.0)) return;
    double tot2 = 0.0;
    for (int k = 0; k < nb; ++k) { h[k] = pow(hist[d * nb + k] / tot, alpha); tot2 += h[k]; }
    const double share = tot2 / nb;
    double acc = 0.0;
    int k = 0;
    ne[0] = ed[0]; ne[nb] = ed[nb];
    for (int j = 1; j < nb; ++j) {
        const double target = share * j;
        while (k < nb - 1 && acc + h[k] < target) { acc += h[k]; ++k; }
        double frac = h[k] > 0.0 ? (target - acc) / h[k] : 0.0;
        if (frac > 1.0) frac = 1.0;
        ne[j] = ed[k] + frac * (ed[k + 1] - ed[k]);
    }
    for (int j = 0; j <= nb; ++j) ed[j] = ne[j];
}

// eq. 1.74, 1.75 (over N - 1) from the sums; eq. 1.82-1.83 over M iterations: res = {Ebar, S2bar, chi2/dof}
__global__ void k_vegas_estimate(long long n, const double *__restrict__ sums, double *__restrict__ res)
{
    if (threadIdx.x || blockIdx.x) return;
    const double mean = sums[0] / (double)n;
    res[0] = mean;
    res[1] = (sums[1] / (double)n - mean * mean) / (double)(n - 1);
}
__global__ void k_vegas_combine(int M, const double *__restrict__ E, const double *__restrict__ S2, double *__restrict__ res)
{
    if (threadIdx.x || blockIdx.x) return;
    double sw = 0.0, swe = 0.0;
    for (int i = 0; i < M; ++i) { sw += 1.0 / S2[i]; swe += E[i] / S2[i]; }
    const double s2 = 1.0 / sw, eb = s2 * swe;
    double c = 0.0;
    for (int i = 0; i < M; ++i) c += (E[i] - eb) * (E[i] - eb) / S2[i];
    res[0] = eb; res[1] = s2; res[2] = M > 1 ? c / (M - 1) : 0.0;
}

// ---- unweighting (L2028-2030) ---------------------------------------------------------------------
// positive doubles order like their bit patterns: the maximum is an integer atomicMax
__global__ void __launch_bounds__(256) k_weight_max(long long n, const double *__restrict__ w, unsigned long long *__restrict__ wmax_bits)
{
    double m = 0.0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const double v = w[e];
        m = v > m ? v : m;
    }
    for (int o = 16; o; o >>= 1) { const double v = __shfl_xor_sync(0xffffffffu, m, o); m = v > m ? v : m; }
    if ((threadIdx.x & 31) == 0 && m > 0.0) atomicMax(wmax_bits, (unsigned long long)__double_as_longlong(m));
}
__global__ void __launch_bounds__(256)
k_unweight(long long n, const double *__restrict__ w, const double *__restrict__ u, const unsigned long long *__restrict__ wmax_bits,
           unsigned char *__restrict__ accept, unsigned long long *__restrict__ count)
{
    const double wmax = __longlong_as_double((long long)*wmax_bits);
    unsigned long long c = 0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n; e += (long long)gridDim.x * blockDim.x) {
        const bool ok = w[e] > u[e] * wmax;
        accept[e] = ok ? 1 : 0;
        c += ok ? 1u : 0u;
    }
    for (int o = 16; o; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if ((threadIdx.x & 31) == 0 && c) atomicAdd(count, c);
}

}  // namespace pdfg
