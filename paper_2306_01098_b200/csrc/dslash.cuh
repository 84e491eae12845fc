// dslash.cuh -- the even-odd HISQ Dslash kernel for sm_100a (rows a2-a5 of SURVEY.md section 8).
//
//   out(x) = sum_mu [ X_mu(x) in(x+mu) - X_mu(x-mu)^+ in(x-mu) + W_mu(x) in(x+3mu) - W_mu(x-3mu)^+ in(x-3mu) ]
//
// One thread owns one output site and NR right-hand sides: each of the 16 links is loaded once into
// registers with 128-bit streaming loads and applied to all NR gathered colour vectors
// ("inner loop over N_inner RHS vectors inside each thread").  More right-hand sides
// than NR are spread over CTAs that run back to back (the paper's N_outer, reuse through L2).
// Neighbour indices and the antiperiodic-t sign are computed arithmetically from the
// site coordinates: no index tables, no ghost cells.  HBM-bound by design; no tensor cores (3x3 complex
// blocks are not a dense contraction).
//
// Internal link layout (written once by hisq_set_links): for field f (0 = fat, 1 = Naik), parity p of
// the site that OWNS the link, and direction mu, one block of Vh*18 reals laid out as planes of
// 16-byte chunks:   fp64: 9 planes of double2 (chunk c = complex entry 3*row+col)
//                   fp32: 4 planes of float4 (entries 2j, 2j+1) followed by 1 plane of float2 (entry 8)
// so a warp reading one chunk of 32 consecutive sites reads 512 contiguous bytes.
// Native field layout: (k, c, h) at ((k*3 + c)*Vh + h) complex (include/hisq.h).
#pragma once
#include "common.cuh"

namespace hisq {

enum { MODE_PLAIN = 0,    // out = D in
       MODE_APPLY_A = 1,  // out = m2*u - D in            and  result[k] = Re<u_k, out_k>     (u = p)
       MODE_RESID = 2 };  // out = v - (m2*u - D in)      and  result[k] = ||out_k||^2        (u = x, v = b)

template <typename T> struct DslashArgs {
    Geom g;
    const T* links;      // internal layout, this precision
    const T* in;         // native, parity 1-par, first RHS of this launch
    T* out;              // native, parity par
    const T* u;          // epilogue operands, native, parity par (MODE 1, 2)
    const T* v;
    double* partial;     // [nrhs_total][ncols]
    unsigned* ticket;
    double* result;      // [nrhs_total], written by the last block
    const int* done;     // if non-null and *done != 0 the kernel returns immediately
    double m2;
    int par;             // parity of the output sites
    int k0;              // global index of the first RHS of this launch (rows of `partial`)
    int nrhs_total;
    int nchunks;         // RHS chunks of NR handled by this launch (consecutive CTAs)
    int slab_blocks;     // CTAs per (tile, t) slab and chunk
    unsigned total_blocks; // CTAs of the whole launch group (epilogue ticket)
    int naik_c14;        // 1: Naik links are stored compressed (14 reals, row f2)
    int t0, tn;          // this launch covers tn owned slices: blockIdx.y = j is slice g.t_lo + t0 + j, plus t_skip for
    PeerPush push;       // MODE_APPLY_A on a partitioned lattice: the last CTA also hands the sums to every rank's mailbox
    int t_skip_at, t_skip;  // j >= t_skip_at (two ranges in one launch: the first and last slices around an interior).
                         // A launch GROUP (the launches that share one ticket) covers every owned slice exactly once
};

// block of (field f, owner parity p, direction mu)
template <typename T>
__device__ __forceinline__ const T* link_block(const T* links, int Vh, int f, int p, int mu)
{
    return links + (size_t)((f * 2 + p) * 4 + mu) * ((size_t)Vh * 18);
}

__device__ __forceinline__ void load_link(const double* blk, int Vh, int h, double (&U)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + h;
#pragma unroll
    for (int c = 0; c < 9; ++c) {
        double2 w = ld_stream(p + (size_t)c * Vh);
        U[2 * c] = w.x;
        U[2 * c + 1] = w.y;
    }
}

__device__ __forceinline__ void load_link(const float* blk, int Vh, int h, float (&U)[18])
{
    const float4* p4 = reinterpret_cast<const float4*>(blk) + h;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        float4 w = ld_stream(p4 + (size_t)j * Vh);
        U[4 * j] = w.x; U[4 * j + 1] = w.y; U[4 * j + 2] = w.z; U[4 * j + 3] = w.w;
    }
    float2 w = ld_stream(reinterpret_cast<const float2*>(blk + (size_t)16 * Vh) + h);
    U[16] = w.x; U[17] = w.y;
}

// Compressed Naik link (row f2): rows 0, 1 and one complex number d are stored (14 reals), row 2 = conj(row0 x row1) * d.
// For W = c U with U in U(3) and c real, d = det(U) / c: SU(3) links (d real) and the U(3)-projected links of the
// HISQ smearing (section 7c) are both covered.
template <typename T> __device__ __forceinline__ void reconstruct_row2(T (&U)[18], T dr, T di)
{
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        const int b = (a + 1) % 3, c = (a + 2) % 3;
        const T re = (U[2 * b] * U[6 + 2 * c] - U[2 * b + 1] * U[6 + 2 * c + 1]) - (U[2 * c] * U[6 + 2 * b] - U[2 * c + 1] * U[6 + 2 * b + 1]);
        const T im = (U[2 * b] * U[6 + 2 * c + 1] + U[2 * b + 1] * U[6 + 2 * c]) - (U[2 * c] * U[6 + 2 * b + 1] + U[2 * c + 1] * U[6 + 2 * b]);
        // (re - i im) (dr + i di)
        U[12 + 2 * a] = fma(re, dr, im * di);
        U[12 + 2 * a + 1] = fma(re, di, -(im * dr));
    }
}

__device__ __forceinline__ void load_link_c14(const double* blk, int Vh, int h, double (&U)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + h;
#pragma unroll
    for (int c = 0; c < 6; ++c) {
        double2 w = ld_stream(p + (size_t)c * Vh);
        U[2 * c] = w.x;
        U[2 * c + 1] = w.y;
    }
    const double2 d = ld_stream(p + (size_t)6 * Vh);
    reconstruct_row2(U, d.x, d.y);
}

__device__ __forceinline__ void load_link_c14(const float* blk, int Vh, int h, float (&U)[18])
{
    const float4* p4 = reinterpret_cast<const float4*>(blk) + h;
#pragma unroll
    for (int j = 0; j < 3; ++j) {
        float4 w = ld_stream(p4 + (size_t)j * Vh);
        U[4 * j] = w.x; U[4 * j + 1] = w.y; U[4 * j + 2] = w.z; U[4 * j + 3] = w.w;
    }
    const float2 d = ld_stream(reinterpret_cast<const float2*>(blk + (size_t)12 * Vh) + h);
    reconstruct_row2(U, d.x, d.y);
}

template <typename T>
__device__ __forceinline__ void load_vec(const T* field, int Vh, int h, T (&v)[6])
{
    using C = typename Vec<T>::c1;
    const C* p = reinterpret_cast<const C*>(field) + h;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        C w = ld_keep(p + (size_t)c * Vh);
        v[2 * c] = w.x;
        v[2 * c + 1] = w.y;
    }
}

// acc += U v
template <typename T> __device__ __forceinline__ void mv_acc(const T (&U)[18], const T (&v)[6], T (&acc)[6])
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const T ur = U[2 * (3 * a + b)], ui = U[2 * (3 * a + b) + 1];
            acc[2 * a] = fma(ur, v[2 * b], acc[2 * a]);
            acc[2 * a] = fma(-ui, v[2 * b + 1], acc[2 * a]);
            acc[2 * a + 1] = fma(ur, v[2 * b + 1], acc[2 * a + 1]);
            acc[2 * a + 1] = fma(ui, v[2 * b], acc[2 * a + 1]);
        }
}

#ifndef HISQ_PDL
#define HISQ_PDL 1   // programmatic dependent launch of the Dslash kernels (dslash_launch_impl.cuh); 0: plain <<< >>> launches
#endif
#ifndef HISQ_F32X2
#define HISQ_F32X2 1   // 1: fp32 complex multiply-adds as packed FFMA2 (fma.rn.f32x2, sm_100+): 2/3 of the FMA issue slots
#endif
#if HISQ_F32X2
// (dx, dy) += (ax, ay) * s   as ONE packed instruction (the scalar rides as a broadcast operand)
__device__ __forceinline__ void fma2(float& dx, float& dy, float ax, float ay, float s)
{
    unsigned long long d, a, b;
    asm("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(dx), "f"(dy));
    asm("mov.b64 %0, {%1, %2};" : "=l"(a) : "f"(ax), "f"(ay));
    asm("mov.b64 %0, {%1, %2};" : "=l"(b) : "f"(s), "f"(s));
    asm("fma.rn.f32x2 %0, %1, %2, %0;" : "+l"(d) : "l"(a), "l"(b));
    asm("mov.b64 {%0, %1}, %2;" : "=f"(dx), "=f"(dy) : "l"(d));
}
// acc += U v:   (re, im) += ur * (vr, vi) + ui * (-vi, vr)
__device__ __forceinline__ void mv_acc(const float (&U)[18], const float (&v)[6], float (&acc)[6])
{
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const float sx = -v[2 * b + 1], sy = v[2 * b];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            fma2(acc[2 * a], acc[2 * a + 1], v[2 * b], v[2 * b + 1], U[2 * (3 * a + b)]);
            fma2(acc[2 * a], acc[2 * a + 1], sx, sy, U[2 * (3 * a + b) + 1]);
        }
    }
}
// acc -= U^dagger v:   (re, im) += (-ur) * (vr, vi) + ui * (-vi, vr)   with u = U_ba
__device__ __forceinline__ void mvdag_sub(const float (&U)[18], const float (&v)[6], float (&acc)[6])
{
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const float sx = -v[2 * b + 1], sy = v[2 * b];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            fma2(acc[2 * a], acc[2 * a + 1], v[2 * b], v[2 * b + 1], -U[2 * (3 * b + a)]);
            fma2(acc[2 * a], acc[2 * a + 1], sx, sy, U[2 * (3 * b + a) + 1]);
        }
    }
}
#endif

// acc -= U^dagger v       ((U^+)_ab = conj(U_ba))
template <typename T> __device__ __forceinline__ void mvdag_sub(const T (&U)[18], const T (&v)[6], T (&acc)[6])
{
#pragma unroll
    for (int a = 0; a < 3; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            const T ur = U[2 * (3 * b + a)], ui = U[2 * (3 * b + a) + 1];
            acc[2 * a] = fma(-ur, v[2 * b], acc[2 * a]);
            acc[2 * a] = fma(-ui, v[2 * b + 1], acc[2 * a]);
            acc[2 * a + 1] = fma(-ur, v[2 * b + 1], acc[2 * a + 1]);
            acc[2 * a + 1] = fma(ui, v[2 * b], acc[2 * a + 1]);
        }
}

// One of the 16 stencil terms for all NR right-hand sides.
//   FWD:  acc += s * F_mu(x) in(x + hop mu)          link owned by the output site (index h, parity par)
//   !FWD: acc -= s * F_mu(x - hop mu)^+ in(x - hop mu) link owned by the neighbour (index hn, parity 1-par)
// s = -1 iff the hop crossed the t boundary (`flip`).  The gathered vectors are loaded VB at a time
// (register budget: 18 reals of link + 6*VB of vectors live beside the 6*NR accumulators).
template <typename T, int NR, int VB, bool FWD>
__device__ __forceinline__ void stencil_term(const T* blk, int hl, const T* in, int Vh, int hn, bool tdir, bool flip, bool c14,
                                             T (&acc)[NR][6])
{
    T U[18];
    if (c14) load_link_c14(blk, Vh, hl, U);
    else load_link(blk, Vh, hl, U);
#if HISQ_SIGN_BRANCH
    if (tdir && flip) {
        // antiperiodic t: the whole CTA shares t (blockIdx.y), so `flip` is block-uniform: a real branch, taken only
        // by the CTAs next to the t boundary, negates the 18 link registers (instead of 6*NR gathered reals)
#pragma unroll
        for (int i = 0; i < 18; ++i) U[i] = -U[i];
    }
#else
    if (tdir) {
        const T sgn = flip ? T(-1) : T(1);
#pragma unroll
        for (int i = 0; i < 18; ++i) U[i] *= sgn;
    }
#endif
#pragma unroll
    for (int k0 = 0; k0 < NR; k0 += VB) {
        T v[VB][6];
#pragma unroll
        for (int j = 0; j < VB; ++j)
            if (k0 + j < NR) load_vec(in + (size_t)(k0 + j) * 3 * 2 * Vh, Vh, hn, v[j]);
#pragma unroll
        for (int j = 0; j < VB; ++j) {
            if (k0 + j < NR) {
                if (FWD) mv_acc(U, v[j], acc[k0 + j]);
                else mvdag_sub(U, v[j], acc[k0 + j]);
            }
        }
    }
}

// NR from which the 8 (mu, hop) pairs run as a real loop of HISQ_ROLL_OUTER trips (the rest unrolled inside): the
// fully unrolled 8-RHS body is > 100 KB of SASS and `no_instruction` became its largest stall (profiles/);
// fp32 gains from rolling, fp64 does not (measured).
#ifndef HISQ_F32_ROLL_FROM
#define HISQ_F32_ROLL_FROM 99
#endif
#ifndef HISQ_F64_ROLL_FROM
#define HISQ_F64_ROLL_FROM 99
#endif
#ifndef HISQ_SIGN_BRANCH
#define HISQ_SIGN_BRANCH 1  // 1: block-uniform branch negates the link at the t boundary; 0: multiply by +-1 always
#endif
// Tuning knobs (measured on B200): vectors gathered per batch and minimum CTAs per SM
// (i.e. the register cap) for the 4-RHS and the 6/8-RHS kernels, per precision.
#ifndef HISQ_ROLL_OUTER
#define HISQ_ROLL_OUTER 2    // trips of the real loop when rolled: 2, 4 or 8
#endif
#ifndef HISQ_F32_VB8
#define HISQ_F32_VB8 8
#endif
#ifndef HISQ_F32_MINB8
#define HISQ_F32_MINB8 4
#endif
#ifndef HISQ_F32_MINB4
#define HISQ_F32_MINB4 6
#endif
#ifndef HISQ_F32_MINB1
#define HISQ_F32_MINB1 3
#endif
#ifndef HISQ_F64_MINB1
#define HISQ_F64_MINB1 4
#endif
#ifndef HISQ_EARLY_MAX
#define HISQ_EARLY_MAX 4   // kernels with NR <= this fetch the epilogue operands before the stencil
#endif
#ifndef HISQ_F32_MINB4_EPI
#define HISQ_F32_MINB4_EPI 4   // register cap of the NR = 3, 4 fp32 kernels WITH an epilogue
#endif
#ifndef HISQ_F32_MINB2
#define HISQ_F32_MINB2 8
#endif
#ifndef HISQ_F64_MINB2
#define HISQ_F64_MINB2 5
#endif
#ifndef HISQ_F64_VB8
#define HISQ_F64_VB8 8
#endif
#ifndef HISQ_F64_MINB8
#define HISQ_F64_MINB8 1
#endif
#ifndef HISQ_F64_MINB4
#define HISQ_F64_MINB4 3
#endif
template <typename T, int NR, int MODE = 0> struct KernelShape {
    static constexpr bool f32 = sizeof(T) == 4;
    static constexpr bool rolled = NR >= (sizeof(T) == 4 ? HISQ_F32_ROLL_FROM : HISQ_F64_ROLL_FROM);
    static constexpr int roll_outer = HISQ_ROLL_OUTER;
    static constexpr int vb8 = f32 ? HISQ_F32_VB8 : HISQ_F64_VB8;
    static constexpr int vb = NR >= 6 ? (vb8 < NR ? vb8 : NR) : NR;
    static constexpr int minb = NR >= 6 ? (f32 ? HISQ_F32_MINB8 : HISQ_F64_MINB8)
                              : NR >= 3 ? (f32 ? (MODE == 0 ? HISQ_F32_MINB4 : HISQ_F32_MINB4_EPI) : HISQ_F64_MINB4)
                              : NR == 2 ? (f32 ? HISQ_F32_MINB2 : HISQ_F64_MINB2) : (f32 ? HISQ_F32_MINB1 : HISQ_F64_MINB1);
};

template <typename T, int NR, int MODE, int BLOCK, bool NC>
__global__ void __launch_bounds__(BLOCK, KernelShape<T, NR, MODE>::minb) dslash_kernel(const DslashArgs<T> a)
{
#if HISQ_PDL
    // let the next kernel of the stream start scheduling its CTAs as this grid's last wave drains, and do not touch
    // memory before everything this launch depends on has completed (programmatic dependent launch, dslash_launch_impl.cuh)
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
    if (a.done != nullptr && *a.done != 0) {
        // solver finished: nothing to compute, but the other ranks' streams still wait for this rank's arrival in
        // the all-reduce of this iteration -- one designated CTA of the launch group keeps the count right
        if (MODE == MODE_APPLY_A && a.push.boxes != nullptr && blockIdx.x == 0 && blockIdx.z == 0 && a.k0 == 0 &&
            (int)blockIdx.y + a.t0 + ((int)blockIdx.y >= a.t_skip_at ? a.t_skip : 0) == a.g.t_cnt - 1)
            peer_push(a.push, a.result, a.nrhs_total);
        return;
    }
    const Geom& g = a.g;
    const int Vh = g.Vh, H = g.H;
    const int chunk = blockIdx.x % a.nchunks;
    const int sc = blockIdx.x / a.nchunks;
    const int trel = (int)blockIdx.y + a.t0 + ((int)blockIdx.y >= a.t_skip_at ? a.t_skip : 0);
    const int t = trel + g.t_lo;
    const int tile = blockIdx.z;
    const int l = sc * BLOCK + threadIdx.x;
    const bool valid = l < H * g.ty * g.tz;

    T acc[NR][6];
#pragma unroll
    for (int k = 0; k < NR; ++k)
#pragma unroll
        for (int i = 0; i < 6; ++i) acc[k][i] = T(0);

    int h = 0;
    const size_t rhs_stride = (size_t)3 * 2 * Vh;  // reals per RHS
    constexpr bool EARLY = MODE != MODE_PLAIN && NR <= HISQ_EARLY_MAX;
    T ue[EARLY ? NR : 1][6], ve[EARLY ? NR : 1][6];
    const T* in = a.in + (size_t)chunk * NR * rhs_stride;
    if (valid) {
        const int xh = l % H;
        const int q = l / H;
        const int yy = q % g.ty, zz = q / g.ty;
        const int y = (tile % g.nty) * g.ty + yy;
        const int z = (tile / g.nty) * g.tz + zz;
        const int par = a.par;
        const int x = 2 * xh + ((par + y + z + t) & 1);
        h = xh + H * (y + g.L[1] * (z + g.L[2] * t));
        const int row = h - xh;
        constexpr int VB = KernelShape<T, NR>::vb;
        if (EARLY) {
            // epilogue operands at the output site are fetched BEFORE the stencil so that their latency hides behind it
            // (a late, dependent load at the end of every CTA cost ~10 % on C2: profiles/r1_launches_bench_c2.md)
#pragma unroll
            for (int k = 0; k < NR; ++k) {
                load_vec(a.u + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, ue[EARLY ? k : 0]);
                if (MODE == MODE_RESID) load_vec(a.v + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, ve[EARLY ? k : 0]);
            }
        }
        if (!KernelShape<T, NR>::rolled) {
            const int c[4] = { x, y, z, t };
            const int stride[4] = { 0, g.sy, g.sz, g.st };
#pragma unroll
            for (int mu = 0; mu < 4; ++mu) {
#pragma unroll
                for (int f = 0; f < 2; ++f) {
                    const int hop = f ? 3 : 1;
                    const int Lmu = g.L[mu];
                    int cp = c[mu] + hop;
                    bool wp = cp >= Lmu;
                    int cm = c[mu] - hop;
                    bool wm = cm < 0;
                    if (mu == 3 && g.part) {   // partitioned in t: read the halo slices, sign only at the global boundary
                        wp = g.flip_hi && cp >= g.t_lo + g.t_cnt;
                        wm = g.flip_lo && cm < g.t_lo;
                    } else {
                        cp -= wp ? Lmu : 0;
                        cm += wm ? Lmu : 0;
                    }
                    int hp, hm;
                    if (mu == 0) { hp = row + (cp >> 1); hm = row + (cm >> 1); }
                    else { hp = h + (cp - c[mu]) * stride[mu]; hm = h + (cm - c[mu]) * stride[mu]; }
                    stencil_term<T, NR, VB, true>(link_block(a.links, Vh, f, par, mu), h, in, Vh, hp, mu == 3, wp, NC && f == 1, acc);
                    stencil_term<T, NR, VB, false>(link_block(a.links, Vh, f, 1 - par, mu), hm, in, Vh, hm, mu == 3, wm, NC && f == 1, acc);
                }
            }
        } else {
            const size_t blk_reals = (size_t)Vh * 18;
            constexpr int NO = KernelShape<T, NR>::roll_outer;   // outer (real) loop trips; 8/NO (mu,hop) pairs unrolled inside
#pragma unroll 1
            for (int o = 0; o < NO; ++o) {
#pragma unroll
                for (int q = 0; q < 8 / NO; ++q) {
                    const int i = o * (8 / NO) + q;
                    const int mu = i >> 1, f = i & 1;
                    const int hop = 1 + 2 * f;
                    const int Lmu = g.L[mu];
                    const int cmu = mu == 0 ? x : (mu == 1 ? y : (mu == 2 ? z : t));
                    int cp = cmu + hop;
                    bool wp = cp >= Lmu;
                    int cm = cmu - hop;
                    bool wm = cm < 0;
                    if (mu == 3 && g.part) {
                        wp = g.flip_hi && cp >= g.t_lo + g.t_cnt;
                        wm = g.flip_lo && cm < g.t_lo;
                    } else {
                        cp -= wp ? Lmu : 0;
                        cm += wm ? Lmu : 0;
                    }
                    // in units of the half-index stride: x counts in pairs (two sites of a row share h)
                    const int u = mu == 0 ? xh : cmu;
                    const int up = mu == 0 ? (cp >> 1) : cp;
                    const int um = mu == 0 ? (cm >> 1) : cm;
                    const int sd = g.stride[mu];
                    const int hp = h + (up - u) * sd, hm = h + (um - u) * sd;
                    const T* lf = a.links + (size_t)((f * 2 + par) * 4 + mu) * blk_reals;
                    const T* lb = a.links + (size_t)((f * 2 + (1 - par)) * 4 + mu) * blk_reals;
                    stencil_term<T, NR, VB, true>(lf, h, in, Vh, hp, mu == 3, wp, NC && f == 1, acc);
                    stencil_term<T, NR, VB, false>(lb, hm, in, Vh, hm, mu == 3, wm, NC && f == 1, acc);
                }
            }
        }
    }

    using C = typename Vec<T>::c1;
    const int kg0 = a.k0 + chunk * NR;  // global index of this thread's first RHS
    double red[NR];
#pragma unroll
    for (int k = 0; k < NR; ++k) red[k] = 0.0;
    if (valid) {
        C* out = reinterpret_cast<C*>(a.out + (size_t)chunk * NR * rhs_stride) + h;
#pragma unroll
        for (int k = 0; k < NR; ++k) {
            T o[6];
            if (MODE == MODE_PLAIN) {
#pragma unroll
                for (int i = 0; i < 6; ++i) o[i] = acc[k][i];
            } else {
                T uu[6];
                if (EARLY) {
#pragma unroll
                    for (int i = 0; i < 6; ++i) uu[i] = ue[EARLY ? k : 0][i];
                } else {
                    load_vec(a.u + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, uu);
                }
                const T m2 = (T)a.m2;
                if (MODE == MODE_APPLY_A) {
#pragma unroll
                    // the 6 products of one site are summed in T and widened once: fp32 -> fp64 conversions run at a
                    // fraction of the FMA rate (12 per RHS and site cost ~25 % of the fp32 n = 4 kernel); sites add in fp64
                    T part = T(0);
                    for (int i = 0; i < 6; ++i) {
                        o[i] = fma(m2, uu[i], -acc[k][i]);
                        part = fma(uu[i], o[i], part);
                    }
                    red[k] += (double)part;
                } else {
                    T vv[6];
                    if (EARLY) {
#pragma unroll
                        for (int i = 0; i < 6; ++i) vv[i] = ve[EARLY ? k : 0][i];
                    } else {
                        load_vec(a.v + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, vv);
                    }
#pragma unroll
                    T part = T(0);
                    for (int i = 0; i < 6; ++i) {
                        o[i] = vv[i] - fma(m2, uu[i], -acc[k][i]);
                        part = fma(o[i], o[i], part);
                    }
                    red[k] += (double)part;
                }
            }
#pragma unroll
            for (int cc = 0; cc < 3; ++cc) {
                C w;
                w.x = o[2 * cc];
                w.y = o[2 * cc + 1];
                out[(size_t)(k * 3 + cc) * Vh] = w;
            }
        }
    }
    if (MODE != MODE_PLAIN) {
        __shared__ double totals[kMaxNrhs];
        const int col = sc + a.slab_blocks * (trel + g.t_cnt * tile);
        const int ncols = a.slab_blocks * g.t_cnt * g.nty * g.ntz;
        if (grid_reduce<NR, BLOCK>(red, kg0, a.partial, ncols, col, a.ticket, a.total_blocks, a.nrhs_total, totals)) {
            if (threadIdx.x < a.nrhs_total) a.result[threadIdx.x] = totals[threadIdx.x];
            if (a.push.boxes) peer_push(a.push, totals, a.nrhs_total);
        }
    }
}

}  // namespace hisq
