// links.cuh -- one-time link repack (row a1 of SURVEY.md section 8): canonical Eq. (5) arrays -> the per-site records the
// Dslash kernel streams (layout: dslash.cuh), and the Naik-link compression test (row f2).
#pragma once
#include "dslash.cuh"

namespace hisq {

// ---- Naik-link compression (row f2; the paper's `CompressionType comp`) -----------------
// A Naik link of the HISQ action is a real multiple of a unitary matrix, W = c U: U in U(3) after the smearing's
// projection (section 7c), in SU(3) for the BASELINE inputs (c = -eta/24).  Store rows 0 and 1 (12 reals) and the complex
// number d = det(W) / |row0 x row1|^2 (= det(U) / c): row 2 = conj(row0 x row1) d.  14 instead of 18 reals per Naik link.
// d and the largest deviation of conj(row0 x row1) d from the stored row 2:
__device__ __forceinline__ double naik_row2_deviation(const double (&e)[18], double& dr, double& di)
{
    double cr[6], det_re = 0.0, det_im = 0.0, c2 = 0.0;   // cr = row0 x row1
    for (int a = 0; a < 3; ++a) {
        const int b = (a + 1) % 3, c = (a + 2) % 3;
        cr[2 * a] = (e[2 * b] * e[6 + 2 * c] - e[2 * b + 1] * e[6 + 2 * c + 1]) - (e[2 * c] * e[6 + 2 * b] - e[2 * c + 1] * e[6 + 2 * b + 1]);
        cr[2 * a + 1] = (e[2 * b] * e[6 + 2 * c + 1] + e[2 * b + 1] * e[6 + 2 * c]) - (e[2 * c] * e[6 + 2 * b + 1] + e[2 * c + 1] * e[6 + 2 * b]);
        det_re += cr[2 * a] * e[12 + 2 * a] - cr[2 * a + 1] * e[12 + 2 * a + 1];
        det_im += cr[2 * a] * e[12 + 2 * a + 1] + cr[2 * a + 1] * e[12 + 2 * a];
        c2 += cr[2 * a] * cr[2 * a] + cr[2 * a + 1] * cr[2 * a + 1];
    }
    dr = c2 > 0.0 ? det_re / c2 : 0.0;
    di = c2 > 0.0 ? det_im / c2 : 0.0;
    double dev = 0.0;
    for (int a = 0; a < 3; ++a) {   // (cr_re - i cr_im) (dr + i di)
        dev = fmax(dev, fabs(cr[2 * a] * dr + cr[2 * a + 1] * di - e[12 + 2 * a]));
        dev = fmax(dev, fabs(cr[2 * a] * di - cr[2 * a + 1] * dr - e[12 + 2 * a + 1]));
    }
    return dev;
}

// Dry run of the compression on the caller's canonical Naik array: counts the links whose row 2 is NOT reproduced to
// `tol` (relative to |row 0|) in the precision the kernels will hold them in; tol32 > 0 additionally tests the values
// rounded to fp32 (HISQ_MIXED keeps an fp32 copy).  The caller compresses only if the count is zero.
template <typename TS>
__global__ void __launch_bounds__(256) naik_check_kernel(const TS* __restrict__ src, int Vh, double tol, double tol32,
                                                         unsigned long long* bad)
{
    const size_t V = (size_t)2 * Vh;
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= 4 * V) return;
    const TS* s = src + idx * 18;
    double e[18];
#pragma unroll
    for (int i = 0; i < 18; ++i) e[i] = (double)s[i];
    double n0 = sqrt(e[0] * e[0] + e[1] * e[1] + e[2] * e[2] + e[3] * e[3] + e[4] * e[4] + e[5] * e[5]);
    double dr, di;
    bool ok = naik_row2_deviation(e, dr, di) <= tol * n0 && n0 > 0.0;
    if (tol32 > 0.0) {
#pragma unroll
        for (int i = 0; i < 18; ++i) e[i] = (double)(float)e[i];
        ok = ok && naik_row2_deviation(e, dr, di) <= tol32 * n0;
    }
    if (!ok) atomicAdd(bad, 1ull);
}

// 18 reals of a canonical link, or (NC) rows 0, 1 and d of its compressed form, as values of TD widened to double
template <typename TS, typename TD, bool NC>
__device__ __forceinline__ int read_link(const TS* __restrict__ s, TD (&o)[18])
{
    if (NC) {
        double e[18];
#pragma unroll
        for (int i = 0; i < 18; ++i) e[i] = (double)(TD)s[i];   // the values the kernel will see
        double dr, di;
        naik_row2_deviation(e, dr, di);
#pragma unroll
        for (int i = 0; i < 12; ++i) o[i] = (TD)e[i];
        o[12] = (TD)dr; o[13] = (TD)di;
        return 14;
    }
#pragma unroll
    for (int i = 0; i < 18; ++i) o[i] = (TD)s[i];
    return 18;
}

// One thread per (site, mu): writes the four links (fat / Naik, forward / backward) of that direction into the site's
// record.  Forward links are the site's own; the backward link of hop h is the link stored at x - h mu (Eq. (5) slot of
// the NEIGHBOUR, opposite parity), fetched here once so that the Dslash never computes a link address again.
// Periodic in all four directions of the context's (for partitioned contexts: extended) lattice.
template <typename TS, typename TD, bool NC>
__global__ void __launch_bounds__(256) link_record_kernel(const TS* __restrict__ fat, const TS* __restrict__ naik,
                                                          TD* __restrict__ dst, const Geom g, size_t nblk)
{
    using R = Rec<TD, NC>;
    const size_t V = (size_t)2 * g.Vh;
    const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;
    if (idx >= 4 * V) return;
    const int mu = (int)(idx / V);
    const size_t eo = idx % V;
    const int par = eo >= (size_t)g.Vh ? 1 : 0;
    const int h = (int)(eo - (size_t)par * g.Vh);
    // coordinates of the site (Eq. (4): lex = 2 h + x-parity bit)
    int q = h;
    const int xh = q % g.H; q /= g.H;
    const int y = q % g.L[1]; q /= g.L[1];
    const int z = q % g.L[2];
    const int t = q / g.L[2];
    int c[4] = { 2 * xh + ((par + y + z + t) & 1), y, z, t };
    TD* rec = dst + (((size_t)par * nblk + (size_t)(h >> 5)) * R::chunks * 32 + (size_t)(h & 31)) * (16 / sizeof(TD));
    constexpr int per = 16 / sizeof(TD);   // reals per chunk: 2 (fp64) or 4 (fp32)
#pragma unroll
    for (int f = 0; f < 2; ++f) {
        const TS* src = f ? naik : fat;
        const int hop = f ? 3 : 1;
        int cn[4] = { c[0], c[1], c[2], c[3] };
        cn[mu] = (c[mu] - hop + g.L[mu]) % g.L[mu];
        const size_t hn = (size_t)(cn[0] >> 1) + (size_t)g.H * (cn[1] + (size_t)g.L[1] * (cn[2] + (size_t)g.L[2] * cn[3]));
        const size_t eo_n = hn + (size_t)(1 - par) * g.Vh;
        TD fw[18], bw[18];
        int nr;
        if (NC && f == 1) {
            nr = read_link<TS, TD, true>(src + ((size_t)mu * V + eo) * 18, fw);
            read_link<TS, TD, true>(src + ((size_t)mu * V + eo_n) * 18, bw);
        } else {
            nr = read_link<TS, TD, false>(src + ((size_t)mu * V + eo) * 18, fw);
            read_link<TS, TD, false>(src + ((size_t)mu * V + eo_n) * 18, bw);
        }
        if (sizeof(TD) == 8) {
            TD* pf = rec + (size_t)R::off(mu * 4 + f * 2) * 32 * per;
            TD* pb = rec + (size_t)R::off(mu * 4 + f * 2 + 1) * 32 * per;
            for (int i = 0; i < nr; ++i) {
                pf[(size_t)(i / per) * 32 * per + i % per] = fw[i];
                pb[(size_t)(i / per) * 32 * per + i % per] = bw[i];
            }
        } else {   // fp32: forward and backward link share the stage, forward first
            TD* pp = rec + (size_t)R::off(mu * 2 + f) * 32 * per;
            for (int i = 0; i < nr; ++i) {
                pp[(size_t)(i / per) * 32 * per + i % per] = fw[i];
                const int j = nr + i;
                pp[(size_t)(j / per) * 32 * per + j % per] = bw[i];
            }
        }
    }
}

}  // namespace hisq
