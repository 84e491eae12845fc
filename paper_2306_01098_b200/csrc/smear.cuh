// smear.cuh -- HISQ link smearing on the GPU: thin links U -> fat links X and Naik links N.
//
//   level 1   V = F7[U]            fat7: c1 = 1/8, c3 = 1/16, c5 = 1/64, c7 = 1/384
//   project   W = V (V^+ V)^(-1/2)
//   level 2   X = F7L[W]           c1 = 1, c3, c5, c7 as above, Lepage -1/8
//             N_mu(x) = W_mu(x) W_mu(x+mu) W_mu(x+2mu)
// ("X and W are smeared gauge fields"; HISQ action, PAPER.md:135 Ref. [53]; reading R26.)
//
// Unlike the oracle (explicit enumeration of the 85 paths of a link), the staples are built RECURSIVELY, the way
// production codes do: with  G_nu[L](x) = U_nu(x) L(x+nu) U_nu(x+mu)^+  +  U_nu(x-nu)^+ L(x-nu) U_nu(x-nu+mu)
//     S3_nu = G_nu[U_mu]          S5_nu,rho = G_rho[S3_nu]          S7_nu,rho,sigma = G_sigma[S5_nu,rho]
//     Lepage_nu = up-part of G_nu[up-part of S3_nu] + down-part of G_nu[down-part of S3_nu]
// 18 launches of one kernel per direction and level instead of 84 path products.  The projection is a Newton iteration
// for the polar factor, X <- (X + X^-+) / 2, not an eigen-decomposition.  The gauge field is periodic in all four
// directions.
// Layouts: the ABI side is the CANONICAL link array of include/hisq.h (matrix of (x, mu) at slot mu*V + eo(x), 9 complex
// row-major, i.e. 144-byte records in fp64).  Read lane by lane such records put every lane of a warp-level load on a
// different cache line (first ncu capture of the staple kernel: DRAM traffic = algorithmic bytes but "Mem Busy" 73 % at
// half the copy bandwidth), so all the work in between runs on a structure-of-arrays copy: entry e of the matrix of
// (x, mu) at complex index (mu*9 + e)*V + eo(x) -- a warp reads 32 consecutive complex numbers per load.  The thin links
// are transposed once on the way in, the three results once on the way out.
#pragma once
#include "common.cuh"

namespace hisq {

template <typename T> struct Mat3 { T r[9], i[9]; };

template <typename T> __device__ __forceinline__ Mat3<T> mat_load(const T* p)
{
    using C = typename Vec<T>::c1;
    const C* q = reinterpret_cast<const C*>(p);
    Mat3<T> m;
#pragma unroll
    for (int e = 0; e < 9; ++e) { const C w = q[e]; m.r[e] = w.x; m.i[e] = w.y; }
    return m;
}
template <typename T> __device__ __forceinline__ void mat_store(T* p, const Mat3<T>& m)
{
    using C = typename Vec<T>::c1;
    C* q = reinterpret_cast<C*>(p);
#pragma unroll
    for (int e = 0; e < 9; ++e) { C w; w.x = m.r[e]; w.y = m.i[e]; q[e] = w; }
}
// structure-of-arrays field of n matrices: entry e of matrix i at complex index e*n + i
template <typename T> __device__ __forceinline__ Mat3<T> soa_load(const T* p, size_t n, size_t i)
{
    using C = typename Vec<T>::c1;
    const C* q = reinterpret_cast<const C*>(p) + i;
    Mat3<T> m;
#pragma unroll
    for (int e = 0; e < 9; ++e) { const C w = q[e * n]; m.r[e] = w.x; m.i[e] = w.y; }
    return m;
}
template <typename T> __device__ __forceinline__ void soa_store(T* p, size_t n, size_t i, const Mat3<T>& m)
{
    using C = typename Vec<T>::c1;
    C* q = reinterpret_cast<C*>(p) + i;
#pragma unroll
    for (int e = 0; e < 9; ++e) { C w; w.x = m.r[e]; w.y = m.i[e]; q[e * n] = w; }
}
template <typename T> __device__ __forceinline__ Mat3<T> mat_add(const Mat3<T>& a, const Mat3<T>& b)
{
    Mat3<T> c;
#pragma unroll
    for (int e = 0; e < 9; ++e) { c.r[e] = a.r[e] + b.r[e]; c.i[e] = a.i[e] + b.i[e]; }
    return c;
}
// DA: use A^+ instead of A; DB: use B^+ instead of B
template <typename T, bool DA, bool DB> __device__ __forceinline__ Mat3<T> mat_mul(const Mat3<T>& a, const Mat3<T>& b)
{
    Mat3<T> c;
#pragma unroll
    for (int i = 0; i < 3; ++i)
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            T sr = T(0), si = T(0);
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                const T ar = DA ? a.r[3 * k + i] : a.r[3 * i + k], ai = DA ? -a.i[3 * k + i] : a.i[3 * i + k];
                const T br = DB ? b.r[3 * j + k] : b.r[3 * k + j], bi = DB ? -b.i[3 * j + k] : b.i[3 * k + j];
                sr = fma(ar, br, sr); sr = fma(-ai, bi, sr);
                si = fma(ar, bi, si); si = fma(ai, br, si);
            }
            c.r[3 * i + j] = sr; c.i[3 * i + j] = si;
        }
    return c;
}

// ---- site arithmetic on the canonical order (Eq. (4)) ----------------------------------------------
struct Site { int c[4]; };
__device__ __forceinline__ Site site_of_eo(const Geom& g, int eo)
{
    const int par = eo >= g.Vh ? 1 : 0;
    const int h = eo - par * g.Vh;
    Site s;
    const int xh = h % g.H;
    int q = h / g.H;
    s.c[1] = q % g.L[1]; q /= g.L[1];
    s.c[2] = q % g.L[2];
    s.c[3] = q / g.L[2];
    s.c[0] = 2 * xh + ((par + s.c[1] + s.c[2] + s.c[3]) & 1);
    return s;
}
__device__ __forceinline__ int eo_of_site(const Geom& g, const Site& s)
{
    const int lex = s.c[0] + g.L[0] * (s.c[1] + g.L[1] * (s.c[2] + g.L[2] * s.c[3]));
    return (lex >> 1) + ((s.c[0] + s.c[1] + s.c[2] + s.c[3]) & 1) * g.Vh;
}
// periodic step of n (|n| <= 3 <= L) in direction d
__device__ __forceinline__ Site hop(const Geom& g, Site s, int d, int n)
{
    int v = s.c[d] + n;
    v = v >= g.L[d] ? v - g.L[d] : (v < 0 ? v + g.L[d] : v);
    s.c[d] = v;
    return s;
}

// ---- out = c1 * U_mu (start of a smeared link) ------------------------------------------------------------------------
template <typename T>
__global__ void __launch_bounds__(128) smear_init_kernel(T* __restrict__ out, const T* __restrict__ in, size_t nreal, T c1)
{
    for (size_t i = (size_t)blockIdx.x * 128 + threadIdx.x; i < nreal; i += (size_t)gridDim.x * 128) out[i] = c1 * in[i];
}

// ---- one generalised staple (see the header): up(x) = U_nu(x) Lu(x+nu) U_nu(x+mu)^+ , dn(x) = U_nu(x-nu)^+ Ld(x-nu) U_nu(x-nu+mu)
// with Lu = a_up (+ b), Ld = a_dn (+ b); acc(x) += coef (up + dn); up / dn are stored to out_up / out_dn if given (their
// sum if both point to the same array).  U: the 4V links being smeared; a_*, b, out_*, acc: V matrices of direction mu.
// All structure-of-arrays (V matrices per block).
constexpr int kStapleMinBlocks = 4;   // CTAs per SM the staple kernel is compiled for (128 registers; measured best of 1, 4, 5, 6)
template <typename T>
__global__ void __launch_bounds__(128, kStapleMinBlocks) staple_kernel(const Geom g, const T* __restrict__ U, const T* __restrict__ a_up,
                                                     const T* __restrict__ a_dn, const T* __restrict__ b, T* out_up, T* out_dn,
                                                     T* __restrict__ acc, int mu, int nu, T coef)
{
    // programmatic dependent launch (as the Dslash kernel): the next launch's CTAs become resident while this grid drains
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int eo = blockIdx.x * 128 + threadIdx.x;
    const size_t V = (size_t)2 * g.Vh;
    if (eo >= (int)V) return;
    const Site x = site_of_eo(g, eo);
    const T* Unu = U + (size_t)nu * V * 18;
    // up
    const int xpn = eo_of_site(g, hop(g, x, nu, 1));
    const int xpm = eo_of_site(g, hop(g, x, mu, 1));
    Mat3<T> L = soa_load(a_up, V, xpn);
    if (b) L = mat_add(L, soa_load(b, V, xpn));
    Mat3<T> up = mat_mul<T, false, true>(mat_mul<T, false, false>(soa_load(Unu, V, eo), L), soa_load(Unu, V, xpm));
    // down
    const Site xm = hop(g, x, nu, -1);
    const int xmn = eo_of_site(g, xm);
    const int xmnpm = eo_of_site(g, hop(g, xm, mu, 1));
    L = soa_load(a_dn, V, xmn);
    if (b) L = mat_add(L, soa_load(b, V, xmn));
    Mat3<T> dn = mat_mul<T, false, false>(mat_mul<T, true, false>(soa_load(Unu, V, xmn), L), soa_load(Unu, V, xmnpm));
    const Mat3<T> sum = mat_add(up, dn);
    if (out_up != nullptr && out_up == out_dn) soa_store(out_up, V, eo, sum);
    else {
        if (out_up) soa_store(out_up, V, eo, up);
        if (out_dn) soa_store(out_dn, V, eo, dn);
    }
    Mat3<T> f = soa_load(acc, V, eo);
#pragma unroll
    for (int e = 0; e < 9; ++e) { f.r[e] = fma(coef, sum.r[e], f.r[e]); f.i[e] = fma(coef, sum.i[e], f.i[e]); }
    soa_store(acc, V, eo, f);
}

// ---- W = V (V^+ V)^(-1/2), in place: Newton iteration for the unitary polar factor, X <- (X + X^-+) / 2 ------------------
// (quadratically convergent for any non-singular V; singular values s -> (s + 1/s)/2).  *bad counts links that did not
// converge (singular or non-finite input).
// links: 4 structure-of-arrays blocks of V matrices.
template <typename T>
__global__ void __launch_bounds__(128) project_u3_kernel(T* __restrict__ links, size_t V, unsigned long long* bad)
{
    const size_t idx = (size_t)blockIdx.x * 128 + threadIdx.x;
    if (idx >= 4 * V) return;
    T* blk = links + (idx / V) * V * 18;
    const size_t site = idx % V;
    Mat3<T> X = soa_load(blk, V, site);
    const T tol = sizeof(T) == 4 ? T(1e-5) : T(1e-12);   // of the LAST step; the error after it is its square
    bool ok = false;
    for (int it = 0; it < 60 && !ok; ++it) {
        // cofactors: inverse = adj / det, adj_ji = cofactor_ij
        Mat3<T> C;
#pragma unroll
        for (int i = 0; i < 3; ++i)
#pragma unroll
            for (int j = 0; j < 3; ++j) {
                const int i1 = (i + 1) % 3, i2 = (i + 2) % 3, j1 = (j + 1) % 3, j2 = (j + 2) % 3;
                const T ar = X.r[3 * i1 + j1], ai = X.i[3 * i1 + j1], br = X.r[3 * i2 + j2], bi = X.i[3 * i2 + j2];
                const T cr = X.r[3 * i1 + j2], ci = X.i[3 * i1 + j2], dr = X.r[3 * i2 + j1], di = X.i[3 * i2 + j1];
                C.r[3 * i + j] = (ar * br - ai * bi) - (cr * dr - ci * di);
                C.i[3 * i + j] = (ar * bi + ai * br) - (cr * di + ci * dr);
            }
        T detr = T(0), deti = T(0);
#pragma unroll
        for (int j = 0; j < 3; ++j) {
            detr += X.r[j] * C.r[j] - X.i[j] * C.i[j];
            deti += X.r[j] * C.i[j] + X.i[j] * C.r[j];
        }
        const T d2 = detr * detr + deti * deti;
        if (!(d2 > T(0)) || !isfinite(d2)) break;
        // X^-1 = C^T / det  =>  X^-+ = conj(C) / conj(det) : element (i,j) = conj(C_ij) / conj(det) = conj(C_ij / det)
        T change = T(0), size = T(0);
#pragma unroll
        for (int e = 0; e < 9; ++e) {
            const T qr = (C.r[e] * detr + C.i[e] * deti) / d2, qi = (C.i[e] * detr - C.r[e] * deti) / d2;   // C_ij / det
            const T nr = T(0.5) * (X.r[e] + qr), ni = T(0.5) * (X.i[e] - qi);
            change += (nr - X.r[e]) * (nr - X.r[e]) + (ni - X.i[e]) * (ni - X.i[e]);
            size += nr * nr + ni * ni;
            X.r[e] = nr; X.i[e] = ni;
        }
        ok = change <= tol * tol * size;
    }
    if (!ok) atomicAdd(bad, 1ull);
    soa_store(blk, V, site, X);
}

// ---- N_mu(x) = scale * eta_mu(x) * W_mu(x) W_mu(x+mu) W_mu(x+2mu)  (W structure-of-arrays, N canonical) ---------------------------------------------------------
__device__ __forceinline__ int eta_sign(const Site& s, int mu)
{
    const int e = mu == 0 ? 0 : (mu == 1 ? s.c[0] : (mu == 2 ? s.c[0] + s.c[1] : s.c[0] + s.c[1] + s.c[2]));
    return 1 - 2 * (e & 1);
}
template <typename T>
__global__ void __launch_bounds__(128) naik_kernel(const Geom g, const T* __restrict__ W, T* __restrict__ out, T scale, int fold)
{
    const int V = 2 * g.Vh;
    const int eo = blockIdx.x * 128 + threadIdx.x;
    const int mu = blockIdx.y;
    if (eo >= V) return;
    const Site x = site_of_eo(g, eo);
    const T* Wm = W + (size_t)mu * V * 18;
    const int x1 = eo_of_site(g, hop(g, x, mu, 1)), x2 = eo_of_site(g, hop(g, x, mu, 2));
    Mat3<T> P = mat_mul<T, false, false>(mat_mul<T, false, false>(soa_load(Wm, V, eo), soa_load(Wm, V, x1)), soa_load(Wm, V, x2));
    const T s = fold ? scale * (T)eta_sign(x, mu) : scale;
#pragma unroll
    for (int e = 0; e < 9; ++e) { P.r[e] *= s; P.i[e] *= s; }
    mat_store(out + ((size_t)mu * V + eo) * 18, P);
}
// ---- layout conversion of a link field (4V matrices), optionally times scale * eta_mu(x) -------------------------------
// TO_SOA: canonical -> structure-of-arrays; else structure-of-arrays -> canonical.  src != dst.
template <typename T, bool TO_SOA>
__global__ void __launch_bounds__(128) link_layout_kernel(const Geom g, const T* __restrict__ src, T* __restrict__ dst, T scale, int fold)
{
    const size_t V = (size_t)2 * g.Vh;
    const int eo = blockIdx.x * 128 + threadIdx.x;
    const int mu = blockIdx.y;
    if (eo >= (int)V) return;
    const T s = fold ? scale * (T)eta_sign(site_of_eo(g, eo), mu) : scale;
    Mat3<T> m = TO_SOA ? mat_load(src + ((size_t)mu * V + eo) * 18) : soa_load(src + (size_t)mu * V * 18, V, eo);
#pragma unroll
    for (int e = 0; e < 9; ++e) { m.r[e] *= s; m.i[e] *= s; }
    if (TO_SOA) soa_store(dst + (size_t)mu * V * 18, V, eo, m);
    else mat_store(dst + ((size_t)mu * V + eo) * 18, m);
}

}  // namespace hisq
