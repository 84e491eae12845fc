// dslash.cuh -- the even-odd HISQ Dslash kernel for sm_100a (rows a2-a5 of SURVEY.md section 8).
//
//   out(x) = sum_mu [ X_mu(x) in(x+mu) - X_mu(x-mu)^+ in(x-mu) + W_mu(x) in(x+3mu) - W_mu(x-3mu)^+ in(x-3mu) ]
//
// One thread owns one output site and NR right-hand sides: each of the 16 links is fetched once and applied to
// all NR gathered colour vectors ("inner loop over N_inner RHS vectors inside each thread").
// More right-hand sides than NR are spread over CTAs that run back to back (the paper's N_outer, reuse through L2).
// Neighbour indices and the antiperiodic-t sign are computed arithmetically from the site
// coordinates: no index tables, no ghost cells.  HBM-bound by design; no tensor cores (3x3 complex blocks are not
// a dense contraction).
//
// Link storage (written once by hisq_set_links): the 16 links an OUTPUT site needs -- its own
// 8 forward links and the 8 links of its backward neighbours, gathered once at set-up time -- form one record; the
// records of 32 consecutive sites (one warp) are interleaved by 16-byte chunk:
//     links[parity][block = h / 32][chunk][lane = h % 32]        (16-byte units)
// so that (1) every link load of a thread is ONE base address plus a compile-time offset (the 16-byte-plane layout of
// round 1 spent ~300 integer instructions per site on link addresses), (2) a warp's loads are 512 contiguous bytes, and
// (3) the data of one stencil term for one warp is one contiguous run of 3.5 - 4.5 KB.  (3) was built for a bulk-copy
// (TMA) link stream -- cp.async.bulk.prefetch.L2 some stages ahead, or cp.async.bulk into a per-warp shared-memory ring
// with mbarriers; both were measured and neither changed the time of any shape (the multi-RHS
// kernels wait for the gathered vectors, not for the links), so plain streaming loads are what ships.
// A STAGE is that run: fp64: one link (9 chunks of double2; compressed Naik link: 7); fp32: the forward and the
// backward link of one (mu, hop) pair (36 floats = 9 chunks of float4; compressed Naik pair: 28 floats = 7).
// Native field layout: (k, c, h) at ((k*3 + c)*Vh + h) complex (include/hisq.h).
#pragma once
#include "common.cuh"

namespace hisq {

enum { MODE_PLAIN = 0,    // out = D in
       MODE_APPLY_A = 1,  // out = m2*u - D in            and  result[k] = Re<u_k, out_k>     (u = p)
       MODE_RESID = 2 };  // out = v - (m2*u - D in)      and  result[k] = ||out_k||^2        (u = x, v = b)

constexpr int kDslashBlock = 128;
constexpr int kDslashWarps = kDslashBlock / 32;
constexpr int kChunkBytes = 512;       // 32 lanes x 16 bytes
constexpr int kStageChunksMax = 9;

template <typename T> struct DslashArgs {
    Geom g;
    const T* links;      // record array of this precision, parity 0 first
    size_t nblk;         // 32-site blocks per parity (records per parity)
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
    // warp -> sites map of one (tile, t) slab: nseg runs of seg_len consecutive half-indices, wps warps each; a warp
    // covers one ALIGNED block of 32 half-indices (lanes outside the run idle: only when seg_len % 32 != 0)
    int nseg, seg_len, wps, merged;
    int wide_dot;        // epilogue scalar products: 1 = every product widened to fp64, 0 = the 6 products of one site summed
                         // in T and widened once (fp32 only matters: fp64 is the same either way)
    int t0, tn;          // this launch covers tn owned slices: blockIdx.y = j is slice g.t_lo + t0 + j, plus t_skip for
    PeerPush push;       // MODE_APPLY_A on a partitioned lattice: the last CTA also hands the sums to every rank's mailbox
    int t_skip_at, t_skip;  // j >= t_skip_at (two ranges in one launch: the first and last slices around an interior).
                         // A launch GROUP (the launches that share one ticket) covers every owned slice exactly once
};

// ---- record layout -------------------------------------------------------------------------------------------------
template <typename T, bool NC> struct Rec {
    static constexpr bool f32 = sizeof(T) == 4;
    static constexpr int nf = 9;                  // chunks of a fat stage
    static constexpr int nn = NC ? 7 : 9;         // chunks of a Naik stage (NC: 14-real compressed links, row f2)
    static constexpr int per_mu = f32 ? (nf + nn) : 2 * (nf + nn);
    static constexpr int chunks = 4 * per_mu;     // per site: fp32 72 / 64, fp64 144 / 128 chunks of 16 bytes
    static constexpr int nstage = f32 ? 8 : 16;
    // stage s: fp32 s = mu*2 + f (both directions); fp64 s = mu*4 + f*2 + dir (dir 0: forward, own link; 1: backward)
    __host__ __device__ static constexpr int off(int s)
    {
        return f32 ? (s >> 1) * per_mu + ((s & 1) ? nf : 0)
                   : (s >> 2) * per_mu + (((s >> 1) & 1) ? 2 * nf + (s & 1) * nn : (s & 1) * nf);
    }
    __host__ __device__ static constexpr int nch(int s) { return (f32 ? (s & 1) : ((s >> 1) & 1)) ? nn : nf; }
};

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

// fp32 complex multiply-adds as packed FFMA2 (fma.rn.f32x2, sm_100+): 2/3 of the FMA issue slots of the scalar form
// (measured: n = 4 573 -> 479 us, n = 8 835-860 -> 790-810 us on 64^3 x 16).
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

// Tuning (measured on B200): vectors gathered per batch and minimum CTAs per SM (i.e. the register
// cap), per precision and RHS count; how the link stream is fetched.
template <typename T, int NR, int MODE = 0> struct KernelShape {
    static constexpr bool f32 = sizeof(T) == 4;
    static constexpr int vb = NR >= 6 ? 4 : NR;   // gathered vectors in flight per stencil term
    static constexpr int minb = NR >= 6 ? (f32 ? 4 : 1)
                              : NR >= 3 ? (f32 ? (MODE == 0 ? 5 : 4) : 3)
                              : NR == 2 ? (f32 ? 8 : 5) : (f32 ? 3 : 4);
    static constexpr bool early = MODE != MODE_PLAIN && NR <= 4;   // fetch the epilogue operands before the stencil
};
// all chunks of stage s of this lane's record
template <typename T, bool NC>
__device__ __forceinline__ void fetch_stage(const typename Vec<T>::c16* rec, int s, typename Vec<T>::c16 (&w)[kStageChunksMax])
{
    using R = Rec<T, NC>;
#pragma unroll
    for (int c = 0; c < kStageChunksMax; ++c)
        if (c < R::nch(s)) w[c] = ld_stream(rec + (R::off(s) + c) * 32);
}

// stage data -> link matrices
__device__ __forceinline__ void unpack_link(const double2 (&w)[kStageChunksMax], bool c14, double (&U)[18])
{
    if (c14) {
#pragma unroll
        for (int c = 0; c < 6; ++c) { U[2 * c] = w[c].x; U[2 * c + 1] = w[c].y; }
        reconstruct_row2(U, w[6].x, w[6].y);
    } else {
#pragma unroll
        for (int c = 0; c < 9; ++c) { U[2 * c] = w[c].x; U[2 * c + 1] = w[c].y; }
    }
}
__device__ __forceinline__ void unpack_pair(const float4 (&w)[kStageChunksMax], bool c14, float (&Uf)[18], float (&Ub)[18])
{
    float e[36];
#pragma unroll
    for (int c = 0; c < 9; ++c) { e[4 * c] = w[c].x; e[4 * c + 1] = w[c].y; e[4 * c + 2] = w[c].z; e[4 * c + 3] = w[c].w; }
    if (c14) {   // 28 floats: forward rows 0, 1 + d, backward rows 0, 1 + d
#pragma unroll
        for (int i = 0; i < 12; ++i) { Uf[i] = e[i]; Ub[i] = e[14 + i]; }
        reconstruct_row2(Uf, e[12], e[13]);
        reconstruct_row2(Ub, e[26], e[27]);
    } else {
#pragma unroll
        for (int i = 0; i < 18; ++i) { Uf[i] = e[i]; Ub[i] = e[18 + i]; }
    }
}

// One stencil term for all NR right-hand sides with the link already in registers.
//   FWD:  acc += s * F_mu(x) in(x + hop mu)            !FWD: acc -= s * F_mu(x - hop mu)^+ in(x - hop mu)
// s = -1 iff the hop crossed the t boundary (`flip`): the whole CTA shares t (blockIdx.y), so `flip` is block-uniform and
// a real branch, taken only by the CTAs next to the t boundary, negates the 18 link registers (not 6*NR gathered reals).
template <typename T, int NR, int VB, bool FWD>
__device__ __forceinline__ void apply_term(T (&U)[18], const T* in, int Vh, int hn, bool tdir, bool flip, T (&acc)[NR][6])
{
    if (tdir && flip) {
#pragma unroll
        for (int i = 0; i < 18; ++i) U[i] = -U[i];
    }
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

template <typename T, int NR, int MODE, bool NC>
__global__ void __launch_bounds__(kDslashBlock, KernelShape<T, NR, MODE>::minb) dslash_kernel(const DslashArgs<T> a)
{
    // programmatic dependent launch: let the next kernel of the stream start scheduling its CTAs as this grid's last wave
    // drains, and do not touch memory before everything this launch depends on has completed (dslash_launch_impl.cuh)
    asm volatile("griddepcontrol.launch_dependents;");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (a.done != nullptr && *a.done != 0) {
        // solver finished: nothing to compute, but the other ranks' streams still wait for this rank's arrival in
        // the all-reduce of this iteration -- one designated CTA of the launch group keeps the count right
        if (MODE == MODE_APPLY_A && a.push.boxes != nullptr && blockIdx.x == 0 && blockIdx.z == 0 && a.k0 == 0 &&
            (int)blockIdx.y + a.t0 + ((int)blockIdx.y >= a.t_skip_at ? a.t_skip : 0) == a.g.t_cnt - 1)
            peer_push(a.push, a.result, a.nrhs_total);
        return;
    }
    using R = Rec<T, NC>;
    using V16 = typename Vec<T>::c16;
    const Geom& g = a.g;
    const int Vh = g.Vh, H = g.H;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int chunk = blockIdx.x % a.nchunks;
    const int sc = blockIdx.x / a.nchunks;
    const int trel = (int)blockIdx.y + a.t0 + ((int)blockIdx.y >= a.t_skip_at ? a.t_skip : 0);
    const int t = trel + g.t_lo;
    const int tile = blockIdx.z;
    // warp -> run of consecutive half-indices -> aligned block of 32
    const int wslab = sc * kDslashWarps + warp;
    const int seg = wslab / a.wps, wseg = wslab - seg * a.wps;
    const bool wvalid = seg < a.nseg;
    const int y0 = (tile % g.nty) * g.ty;
    const int z0 = g.z_lo + (tile / g.nty) * g.tz + (a.merged ? 0 : seg);
    const int hseg = H * (y0 + g.L[1] * (z0 + g.L[2] * t));
    const int hb = (hseg >> 5) + wseg;
    const bool valid = wvalid && hb * 32 + lane >= hseg && hb * 32 + lane < hseg + a.seg_len;
    const int h = valid ? hb * 32 + lane : hseg;   // idle lanes of a live warp compute on a valid site and store nothing

    T acc[NR][6];
#pragma unroll
    for (int k = 0; k < NR; ++k)
#pragma unroll
        for (int i = 0; i < 6; ++i) acc[k][i] = T(0);

    const size_t rhs_stride = (size_t)3 * 2 * Vh;  // reals per RHS
    constexpr bool EARLY = KernelShape<T, NR, MODE>::early;
    T ue[EARLY ? NR : 1][6], ve[EARLY ? NR : 1][6];
    const T* in = a.in + (size_t)chunk * NR * rhs_stride;
    if (wvalid) {
        const int par = a.par;
        const V16* rec = reinterpret_cast<const V16*>(a.links) + ((size_t)par * a.nblk + hb) * ((size_t)R::chunks * 32) + lane;
        const int rel = h - hseg;
        const int xh = rel % H;
        const int ry = rel / H;
        const int y = a.merged ? ry % g.L[1] : y0 + ry;
        const int z = a.merged ? z0 + ry / g.L[1] : z0;
        const int x = 2 * xh + ((par + y + z + t) & 1);
        const int row = h - xh;
        constexpr int VB = KernelShape<T, NR, MODE>::vb;
        if (EARLY) {
            // epilogue operands at the output site are fetched BEFORE the stencil so that their latency hides behind it
#pragma unroll
            for (int k = 0; k < NR; ++k) {
                load_vec(a.u + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, ue[EARLY ? k : 0]);
                if (MODE == MODE_RESID) load_vec(a.v + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, ve[EARLY ? k : 0]);
            }
        }
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
                } else if (mu == 2 && g.zpart) {   // partitioned in z: read the halo planes (periodic direction: no sign)
                    wp = wm = false;
                } else {
                    cp -= wp ? Lmu : 0;
                    cm += wm ? Lmu : 0;
                }
                int hp, hm;
                if (mu == 0) { hp = row + (cp >> 1); hm = row + (cm >> 1); }
                else { hp = h + (cp - c[mu]) * stride[mu]; hm = h + (cm - c[mu]) * stride[mu]; }
                V16 w[kStageChunksMax];
                if (sizeof(T) == 4) {
                    const int s = mu * 2 + f;
                    fetch_stage<T, NC>(rec, s, w);
                    T Uf[18], Ub[18];
                    unpack_pair(reinterpret_cast<const float4(&)[kStageChunksMax]>(w), NC && f == 1,
                                reinterpret_cast<float(&)[18]>(Uf), reinterpret_cast<float(&)[18]>(Ub));
                    apply_term<T, NR, VB, true>(Uf, in, Vh, hp, mu == 3, wp, acc);
                    apply_term<T, NR, VB, false>(Ub, in, Vh, hm, mu == 3, wm, acc);
                } else {
                    const int s = mu * 4 + f * 2;
                    T U[18];
                    fetch_stage<T, NC>(rec, s, w);
                    unpack_link(reinterpret_cast<const double2(&)[kStageChunksMax]>(w), NC && f == 1, reinterpret_cast<double(&)[18]>(U));
                    apply_term<T, NR, VB, true>(U, in, Vh, hp, mu == 3, wp, acc);
                    fetch_stage<T, NC>(rec, s + 1, w);
                    unpack_link(reinterpret_cast<const double2(&)[kStageChunksMax]>(w), NC && f == 1, reinterpret_cast<double(&)[18]>(U));
                    apply_term<T, NR, VB, false>(U, in, Vh, hm, mu == 3, wm, acc);
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
                    // a.wide_dot == 0: the 6 products of one site are summed in T and widened once: fp32 -> fp64 conversions
                    // run at a fraction of the FMA rate (12 per RHS and site cost ~25 % of the fp32 n = 4 kernel); sites add
                    // in fp64 either way.  The launcher widens every product where the kernel is DRAM-bound anyway (NR <= 2).
                    T part = T(0);
                    double wide = 0.0;
#pragma unroll
                    for (int i = 0; i < 6; ++i) {
                        o[i] = fma(m2, uu[i], -acc[k][i]);
                        if (sizeof(T) == 4 && a.wide_dot) wide = fma((double)uu[i], (double)o[i], wide);
                        else part = fma(uu[i], o[i], part);
                    }
                    red[k] += (sizeof(T) == 4 && a.wide_dot) ? wide : (double)part;
                } else {
                    T vv[6];
                    if (EARLY) {
#pragma unroll
                        for (int i = 0; i < 6; ++i) vv[i] = ve[EARLY ? k : 0][i];
                    } else {
                        load_vec(a.v + (size_t)(chunk * NR + k) * rhs_stride, Vh, h, vv);
                    }
                    T part = T(0);
                    double wide = 0.0;
#pragma unroll
                    for (int i = 0; i < 6; ++i) {
                        o[i] = vv[i] - fma(m2, uu[i], -acc[k][i]);
                        if (sizeof(T) == 4 && a.wide_dot) wide = fma((double)o[i], (double)o[i], wide);
                        else part = fma(o[i], o[i], part);
                    }
                    red[k] += (sizeof(T) == 4 && a.wide_dot) ? wide : (double)part;
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
        if (grid_reduce<NR, kDslashBlock>(red, kg0, a.partial, ncols, col, a.ticket, a.total_blocks, a.nrhs_total, totals)) {
            if (threadIdx.x < a.nrhs_total) a.result[threadIdx.x] = totals[threadIdx.x];
            if (a.push.boxes) peer_push(a.push, totals, a.nrhs_total);
        }
    }
}

}  // namespace hisq
