// pb_device.cuh -- device-side building blocks shared by the hot kernels: TMA bulk copies with
// mbarrier completion (sm_100a), and the fp64 rsqrt / exp(-kappa r) used per interaction.
// Product code.  Nothing here includes, links or calls anything under oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

// ---- TMA 1-D bulk copy global -> shared, completion on an mbarrier --------------------------------
__device__ __forceinline__ uint32_t pb_smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void pb_mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(pb_smem_u32(bar)), "r"(count) : "memory");
}

__device__ __forceinline__ void pb_mbar_fence_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}

__device__ __forceinline__ void pb_mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(pb_smem_u32(bar)), "r"(bytes) : "memory");
}

__device__ __forceinline__ void pb_mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(pb_smem_u32(bar)) : "memory");
}

// bytes must be a multiple of 16, src and dst 16-byte aligned
__device__ __forceinline__ void pb_bulk_g2s(void* dst, const void* src, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     pb_smem_u32(dst)),
                 "l"(src), "r"(bytes), "r"(pb_smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ void pb_mbar_wait(uint64_t* bar, uint32_t parity)
{
    uint32_t ok;
    const uint32_t a = pb_smem_u32(bar);
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok)
            : "r"(a), "r"(parity)
            : "memory");
    } while (!ok);
}

// ---- per-interaction arithmetic ---------------------------------------------------------------------
// Constants of exp(-kappa r) (filled on the host by pb_make_expk, passed by value):
//   n = rint(r * c1), c1 = 32 kappa / ln 2;  g = r - n * Lk, Lk = ln 2 / (32 kappa), |kappa g| <= ln2/64;
//   exp(-kappa r) = 2^-(n>>5) * T[n&31] * sum_{m<=6} c[m] g^m,  c[m] = (-kappa)^m / m!,  T[j] = 2^(-j/32).
// Truncation error (kappa g)^7/7! < 4e-18; the result is good to ~3e-16 relative (D: R-29).
struct pb_expk {
    double c1, Lk;
    double c[7];
    double T[32];
    double g[12];     // g[m] = kappa^2 / ((2m+1)(2m-1)): the Yukawa radial recurrence with the layers scaled by (2m-1)!! (m2p_radial)
};

// Finer table, shorter polynomial, for the P2P kernel where exp(-kappa r) is evaluated once per pair:
//   n = rint(r * c1), c1 = 256 kappa / ln 2;  g = r - n * Lk, |kappa g| <= ln2/512;
//   exp(-kappa r) = 2^-(n>>8) * T256[n&255] * sum_{m<=4} c[m] g^m      (truncation (kappa g)^5/5! < 4e-17)
struct pb_expk8 {
    double c1, Lk;
    double c[5];
};

__device__ __forceinline__ double pb_exp_mkr8(double r, const pb_expk8& k, const double* __restrict__ T256)
{
    const double MAGIC = 6755399441055744.0;   // 1.5 * 2^52: the low word of (v + MAGIC) is rint(v)
    const double s = fma(r, k.c1, MAGIC);
    const double nf = s - MAGIC;
    const double g = fma(nf, -k.Lk, r);
    unsigned n = (unsigned)__double2loint(s);
    n = n < 256000u ? n : 256000u;              // exp(-690) already underflows; also tames padding lanes
    double p = k.c[4];
    p = fma(p, g, k.c[3]);
    p = fma(p, g, k.c[2]);
    p = fma(p, g, k.c[1]);
    p = fma(p, g, k.c[0]);
    const double v = p * T256[n & 255u];
    return __hiloint2double(__double2hiint(v) - (int)((n >> 8) << 20), __double2loint(v));
}

// 1/sqrt(x) for normal positive x: MUFU.RSQ64H seed (~2^-22) and one third-order step
//   e = 1 - x y^2,  y <- y + y e (1/2 + 3/8 e)        (error ~ 0.3 e^3 < 2^-60 before rounding)
__device__ __forceinline__ double pb_rsqrt(double x)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double xy = x * y;
    const double e = fma(-xy, y, 1.0);
    const double q = fma(0.375, e, 0.5);
    const double ye = y * e;
    return fma(ye, q, y);
}

// exp(-kappa r), r >= 0, with the exponent table Ts (32 doubles, shared memory)
__device__ __forceinline__ double pb_exp_mkr(double r, const pb_expk& k, const double* __restrict__ Ts)
{
    const double MAGIC = 6755399441055744.0;   // 1.5 * 2^52: the low word of (v + MAGIC) is rint(v)
    const double s = fma(r, k.c1, MAGIC);
    const double nf = s - MAGIC;
    const double g = fma(nf, -k.Lk, r);
    unsigned n = (unsigned)__double2loint(s);
    n = n < 32000u ? n : 32000u;                // exp(-690) already underflows; also tames padding lanes
    double p = k.c[6];
    p = fma(p, g, k.c[5]);
    p = fma(p, g, k.c[4]);
    p = fma(p, g, k.c[3]);
    p = fma(p, g, k.c[2]);
    p = fma(p, g, k.c[1]);
    p = fma(p, g, k.c[0]);
    const double v = p * Ts[n & 31u];
    return __hiloint2double(__double2hiint(v) - (int)((n >> 5) << 20), __double2loint(v));
}
