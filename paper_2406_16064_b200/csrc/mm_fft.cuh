// mm_fft.cuh — shared-memory FFT core of the demag convolution ("three forward
// Fourier transforms and three inverse Fourier transforms").
//
// Tile model.  A CTA holds a tile of `nlines` independent lines of `n` complex points in shared
// memory, element (point q, line l) at s[q*pitch + l] — the LINE index is the fastest one, so the
// threads of a warp work on the same butterfly of neighbouring lines: every shared-memory access
// of a stage is unit-stride across the warp (bank-conflict free for any radix and any stage) and
// the twiddle factor is warp-uniform.
//
// Transform.  Forward = in-place decimation-in-frequency (Gentleman-Sande), radix 8/4/2, natural
// order in, BIT-REVERSED order out.  Inverse = the exact adjoint, decimation-in-time, bit-reversed
// in, natural out, unnormalised.  Nothing is ever re-ordered: the spectrum lives in bit-reversed
// positions everywhere (HBM included) and the cached tensor spectrum K^ is permuted once at setup.
//
// Zero padding / cropping (R3) are pruned stages: a line of n = 2m points
// whose upper half is zero enters as  s[i] = a_i, s[i+m] = a_i w_n^i  (the first radix-2 DIF stage
// with the zeros folded in) followed by the stages of two independent length-m blocks; the
// cropped inverse ends with  out_i = s[i] + conj(w_n^i) s[i+m], i < m.
//
// Everything here is __host__ __device__ so the index arithmetic can be exercised on the CPU
// (thread loops run with tid = 0, nthr = 1; MM_SYNC is a no-op there).
#pragma once

#if defined(__CUDACC__)
#define MM_HD __host__ __device__ __forceinline__
#else
#define MM_HD inline
#endif

#if defined(__CUDA_ARCH__)
#define MM_SYNC() __syncthreads()
#else
#define MM_SYNC() ((void)0)
#endif

namespace mm {

template <typename T> struct alignas(2 * sizeof(T)) cx {
    T x, y;
};

template <typename T> MM_HD cx<T> mk(T a, T b) { cx<T> r; r.x = a; r.y = b; return r; }

#if defined(__CUDA_ARCH__) && !defined(MM_NO_F32X2)
// sm_100a packed fp32 arithmetic (add/mul/fma.rn.f32x2 -> FADD2 / FMUL2 / FFMA2): one instruction
// per complex add, two per complex multiply.  A complex number is the register pair (re, im); ptxas
// folds the swaps, broadcasts and sign patterns below into operand modifiers of the packed
// instructions, so none of the pack / unpack moves survive into SASS.
#define MM_F32X2 1
typedef unsigned long long mm_u64;
__device__ __forceinline__ mm_u64 pk2(float lo, float hi) { mm_u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ cx<float> upk2(mm_u64 v) { cx<float> r; asm("mov.b64 {%0,%1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v)); return r; }
__device__ __forceinline__ mm_u64 add2(mm_u64 a, mm_u64 b) { mm_u64 r; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ mm_u64 sub2(mm_u64 a, mm_u64 b) { mm_u64 r; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ mm_u64 mul2(mm_u64 a, mm_u64 b) { mm_u64 r; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b)); return r; }
__device__ __forceinline__ mm_u64 fma2(mm_u64 a, mm_u64 b, mm_u64 c) { mm_u64 r; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c)); return r; }
__device__ __forceinline__ cx<float> operator+(cx<float> a, cx<float> b) { return upk2(add2(pk2(a.x, a.y), pk2(b.x, b.y))); }
__device__ __forceinline__ cx<float> operator-(cx<float> a, cx<float> b) { return upk2(sub2(pk2(a.x, a.y), pk2(b.x, b.y))); }
__device__ __forceinline__ cx<float> cmul(cx<float> a, cx<float> b)
{
    return upk2(fma2(pk2(a.y, a.x), pk2(-b.y, b.y), mul2(pk2(a.x, a.y), pk2(b.x, b.x))));
}
__device__ __forceinline__ cx<float> cmulc(cx<float> a, cx<float> b)
{
    return upk2(fma2(pk2(a.y, a.x), pk2(b.y, -b.y), mul2(pk2(a.x, a.y), pk2(b.x, b.x))));
}
__device__ __forceinline__ cx<float> scale(cx<float> a, float s) { return upk2(mul2(pk2(a.x, a.y), pk2(s, s))); }
// a*ka + b*kb (+ c*kc), real coefficients
__device__ __forceinline__ cx<float> lin2(cx<float> a, float ka, cx<float> b, float kb)
{
    return upk2(fma2(pk2(b.x, b.y), pk2(kb, kb), mul2(pk2(a.x, a.y), pk2(ka, ka))));
}
__device__ __forceinline__ cx<float> lin3(cx<float> a, float ka, cx<float> b, float kb, cx<float> c, float kc)
{
    return upk2(fma2(pk2(c.x, c.y), pk2(kc, kc), fma2(pk2(b.x, b.y), pk2(kb, kb), mul2(pk2(a.x, a.y), pk2(ka, ka)))));
}
#endif
template <typename T> MM_HD cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.x + b.x, a.y + b.y); }
template <typename T> MM_HD cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.x - b.x, a.y - b.y); }
template <typename T> MM_HD cx<T> cmul(cx<T> a, cx<T> b) { return mk<T>(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// a * conj(b)
template <typename T> MM_HD cx<T> cmulc(cx<T> a, cx<T> b) { return mk<T>(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y); }
template <typename T> MM_HD cx<T> conj(cx<T> a) { return mk<T>(a.x, -a.y); }
template <typename T> MM_HD cx<T> mul_mi(cx<T> a) { return mk<T>(a.y, -a.x); }   // * (-i)
template <typename T> MM_HD cx<T> mul_pi(cx<T> a) { return mk<T>(-a.y, a.x); }   // * (+i)
template <typename T> MM_HD cx<T> scale(cx<T> a, T s) { return mk<T>(a.x * s, a.y * s); }
template <typename T> MM_HD cx<T> lin2(cx<T> a, T ka, cx<T> b, T kb) { return mk<T>(ka * a.x + kb * b.x, ka * a.y + kb * b.y); }
template <typename T> MM_HD cx<T> lin3(cx<T> a, T ka, cx<T> b, T kb, cx<T> c, T kc)
{
    return mk<T>(ka * a.x + kb * b.x + kc * c.x, ka * a.y + kb * b.y + kc * c.y);
}
template <typename T> MM_HD void bf2(cx<T>& a, cx<T>& b) { cx<T> t = a; a = t + b; b = t - b; }

MM_HD int ilog2(int n) { int l = 0; while ((1 << l) < n) l++; return l; }
// bit reversal of v within `bits` bits
MM_HD unsigned brev(unsigned v, int bits)
{
#if defined(__CUDA_ARCH__)
    return bits ? (__brev(v) >> (32 - bits)) : 0u;
#else
    unsigned r = 0;
    for (int b = 0; b < bits; b++) r |= ((v >> b) & 1u) << (bits - 1 - b);
    return r;
#endif
}

// ---- radix kernels: forward = natural in, bit-reversed out; inverse = the adjoint -------------
template <typename T, int R> struct radix;

template <typename T> struct radix<T, 2> {
    static MM_HD void fwd(cx<T>* v) { bf2(v[0], v[1]); }
    static MM_HD void inv(cx<T>* v) { bf2(v[0], v[1]); }
};
template <typename T> struct radix<T, 4> {
    static MM_HD void fwd(cx<T>* v)
    {
        bf2(v[0], v[2]); bf2(v[1], v[3]); v[3] = mul_mi(v[3]);
        bf2(v[0], v[1]); bf2(v[2], v[3]);
    }
    static MM_HD void inv(cx<T>* v)
    {
        bf2(v[0], v[1]); bf2(v[2], v[3]);
        v[3] = mul_pi(v[3]); bf2(v[0], v[2]); bf2(v[1], v[3]);
    }
};
template <typename T> struct radix<T, 8> {
    static MM_HD void fwd(cx<T>* v)
    {
        const T c = (T)0.70710678118654752440;
#pragma unroll
        for (int r = 0; r < 4; r++) bf2(v[r], v[r + 4]);
        v[5] = mk<T>(c * (v[5].x + v[5].y), c * (v[5].y - v[5].x));      // * (1-i)/sqrt2
        v[6] = mul_mi(v[6]);
        v[7] = mk<T>(c * (v[7].y - v[7].x), -c * (v[7].x + v[7].y));     // * (-1-i)/sqrt2
        radix<T, 4>::fwd(v);
        radix<T, 4>::fwd(v + 4);
    }
    static MM_HD void inv(cx<T>* v)
    {
        const T c = (T)0.70710678118654752440;
        radix<T, 4>::inv(v);
        radix<T, 4>::inv(v + 4);
        v[5] = mk<T>(c * (v[5].x - v[5].y), c * (v[5].x + v[5].y));      // * (1+i)/sqrt2
        v[6] = mul_pi(v[6]);
        v[7] = mk<T>(-c * (v[7].x + v[7].y), c * (v[7].x - v[7].y));     // * (-1+i)/sqrt2
#pragma unroll
        for (int r = 0; r < 4; r++) bf2(v[r], v[r + 4]);
    }
};

// Twiddle table: tw[k] = exp(-2 pi i k / twN), k in [0, twN/2]; generated in fp64, rounded once.
template <typename T> struct twiddles {
    const cx<T>* tw;
    int twN;
    // w_L^i for i < L/2 (L divides twN)
    MM_HD cx<T> get(int i, int L) const { return tw[i * (twN / L)]; }
};

// powers w^0..w^(R-1) stored in bit-reversed slot order: pw[r] = w^{brev(r)}
template <typename T, int R> MM_HD void twiddle_powers(cx<T> w1, cx<T>* pw)
{
    if (R == 2) { pw[1] = w1; }
    else if (R == 4) {
        cx<T> w2 = cmul(w1, w1);
        pw[1] = w2; pw[2] = w1; pw[3] = cmul(w2, w1);
    } else {
        cx<T> w2 = cmul(w1, w1), w3 = cmul(w2, w1), w4 = cmul(w2, w2);
        pw[1] = w4; pw[2] = w2; pw[3] = cmul(w3, w3); pw[4] = w1; pw[5] = cmul(w4, w1); pw[6] = w3; pw[7] = cmul(w4, w3);
    }
}

// One forward radix-R DIF stage on blocks of current length Lc, all lines of the tile.
template <typename T, int R>
MM_HD void dif_stage(cx<T>* s, int pitch, int nlines, int n, int Lc, twiddles<T> tw, int tid, int nthr)
{
    const int sub = Lc / R;
    const int total = (n / R) * nlines;
    for (int f = tid; f < total; f += nthr) {
        const int l = f % nlines, b = f / nlines;
        const int blk = b / sub, i = b - blk * sub;
        cx<T>* p = s + (size_t)(blk * Lc + i) * pitch + l;
        cx<T> v[R];
#pragma unroll
        for (int r = 0; r < R; r++) v[r] = p[(size_t)r * sub * pitch];
        radix<T, R>::fwd(v);
        if (i != 0) {
            cx<T> pw[R];
            twiddle_powers<T, R>(tw.get(i, Lc), pw);
#pragma unroll
            for (int r = 1; r < R; r++) v[r] = cmul(v[r], pw[r]);
        }
#pragma unroll
        for (int r = 0; r < R; r++) p[(size_t)r * sub * pitch] = v[r];
    }
}

// The adjoint stage (inverse DIT), unnormalised.
template <typename T, int R>
MM_HD void dit_stage(cx<T>* s, int pitch, int nlines, int n, int Lc, twiddles<T> tw, int tid, int nthr)
{
    const int sub = Lc / R;
    const int total = (n / R) * nlines;
    for (int f = tid; f < total; f += nthr) {
        const int l = f % nlines, b = f / nlines;
        const int blk = b / sub, i = b - blk * sub;
        cx<T>* p = s + (size_t)(blk * Lc + i) * pitch + l;
        cx<T> v[R];
#pragma unroll
        for (int r = 0; r < R; r++) v[r] = p[(size_t)r * sub * pitch];
        if (i != 0) {
            cx<T> pw[R];
            twiddle_powers<T, R>(tw.get(i, Lc), pw);
#pragma unroll
            for (int r = 1; r < R; r++) v[r] = cmulc(v[r], pw[r]);
        }
        radix<T, R>::inv(v);
#pragma unroll
        for (int r = 0; r < R; r++) p[(size_t)r * sub * pitch] = v[r];
    }
}

// Radix schedule for a block length m: 8 while >= 8, then the remainder (4 or 2).
MM_HD int next_radix(int Lc) { return Lc >= 8 ? 8 : Lc; }

// Forward transform of every length-m block of the n-point lines (n a multiple of m).
template <typename T>
MM_HD void fft_fwd_blocks(cx<T>* s, int pitch, int nlines, int n, int m, twiddles<T> tw, int tid, int nthr)
{
    int Lc = m;
    while (Lc > 1) {
        const int R = next_radix(Lc);
        if (R == 8) dif_stage<T, 8>(s, pitch, nlines, n, Lc, tw, tid, nthr);
        else if (R == 4) dif_stage<T, 4>(s, pitch, nlines, n, Lc, tw, tid, nthr);
        else dif_stage<T, 2>(s, pitch, nlines, n, Lc, tw, tid, nthr);
        MM_SYNC();
        Lc /= R;
    }
}

// Inverse (adjoint) of fft_fwd_blocks: stages in reverse order.
template <typename T>
MM_HD void fft_inv_blocks(cx<T>* s, int pitch, int nlines, int n, int m, twiddles<T> tw, int tid, int nthr)
{
    // the forward schedule is 8,8,...,8,rem ; walk it backwards
    int rem = m;
    while (rem >= 8) rem /= 8;           // rem in {1,2,4}
    int Lc = rem;
    if (rem > 1) {
        if (rem == 4) dit_stage<T, 4>(s, pitch, nlines, n, 4, tw, tid, nthr);
        else dit_stage<T, 2>(s, pitch, nlines, n, 2, tw, tid, nthr);
        MM_SYNC();
    }
    while (Lc < m) {
        Lc *= 8;
        dit_stage<T, 8>(s, pitch, nlines, n, Lc, tw, tid, nthr);
        MM_SYNC();
    }
}

}  // namespace mm

// ================================================================================================
// v2 building blocks: V-wide column vectors (16-byte shared/global accesses for fp32), radix
// kernels on any element type, shift/mask index arithmetic.
// ================================================================================================
namespace mm {

template <typename T, int V> struct alignas(V * 2 * sizeof(T)) cvec {
    cx<T> e[V];
};
template <typename T, int V> MM_HD cvec<T, V> operator+(cvec<T, V> a, cvec<T, V> b)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = a.e[k] + b.e[k];
    return r;
}
template <typename T, int V> MM_HD cvec<T, V> operator-(cvec<T, V> a, cvec<T, V> b)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = a.e[k] - b.e[k];
    return r;
}
template <typename T, int V> MM_HD cvec<T, V> cmul(cvec<T, V> a, cx<T> w)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = cmul(a.e[k], w);
    return r;
}
template <typename T, int V> MM_HD cvec<T, V> cmulc(cvec<T, V> a, cx<T> w)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = cmulc(a.e[k], w);
    return r;
}
template <typename T, int V> MM_HD cvec<T, V> mul_mi(cvec<T, V> a)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = mul_mi(a.e[k]);
    return r;
}
template <typename T, int V> MM_HD cvec<T, V> mul_pi(cvec<T, V> a)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = mul_pi(a.e[k]);
    return r;
}
// multiplication by a compile-time-known constant (c + i s)
template <typename T> MM_HD cx<T> crot(cx<T> a, T c, T s)
{
#if defined(MM_F32X2)
    if (sizeof(T) == 4) return cmul(a, mk<T>(c, s));
#endif
    return mk<T>(c * a.x - s * a.y, c * a.y + s * a.x);
}
template <typename T, int V> MM_HD cvec<T, V> crot(cvec<T, V> a, T c, T s)
{
    cvec<T, V> r;
#pragma unroll
    for (int k = 0; k < V; k++) r.e[k] = crot(a.e[k], c, s);
    return r;
}
template <typename T> struct scalar_of;
template <typename T> struct scalar_of<cx<T>> { typedef T type; };
template <typename T, int V> struct scalar_of<cvec<T, V>> { typedef T type; };

template <typename E> MM_HD void bfe(E& a, E& b) { E t = a; a = t + b; b = t - b; }

// Radix kernels on element type E (cx<T> or cvec<T,V>): fwd = natural in, bit-reversed out; inv = adjoint.
template <typename E, int R> struct rad;
template <typename E> struct rad<E, 1> {
    static MM_HD void fwd(E*) {}
    static MM_HD void inv(E*) {}
};
template <typename E> struct rad<E, 2> {
    static MM_HD void fwd(E* v) { bfe(v[0], v[1]); }
    static MM_HD void inv(E* v) { bfe(v[0], v[1]); }
};
template <typename E> struct rad<E, 4> {
    static MM_HD void fwd(E* v)
    {
        bfe(v[0], v[2]); bfe(v[1], v[3]); v[3] = mul_mi(v[3]);
        bfe(v[0], v[1]); bfe(v[2], v[3]);
    }
    static MM_HD void inv(E* v)
    {
        bfe(v[0], v[1]); bfe(v[2], v[3]);
        v[3] = mul_pi(v[3]); bfe(v[0], v[2]); bfe(v[1], v[3]);
    }
};
template <typename E> struct rad<E, 8> {
    typedef typename scalar_of<E>::type T;
    static MM_HD void fwd(E* v)
    {
        const T c = (T)0.70710678118654752440;
#pragma unroll
        for (int r = 0; r < 4; r++) bfe(v[r], v[r + 4]);
        v[5] = crot(v[5], c, -c); v[6] = mul_mi(v[6]); v[7] = crot(v[7], -c, -c);
        rad<E, 4>::fwd(v); rad<E, 4>::fwd(v + 4);
    }
    static MM_HD void inv(E* v)
    {
        const T c = (T)0.70710678118654752440;
        rad<E, 4>::inv(v); rad<E, 4>::inv(v + 4);
        v[5] = crot(v[5], c, c); v[6] = mul_pi(v[6]); v[7] = crot(v[7], -c, c);
#pragma unroll
        for (int r = 0; r < 4; r++) bfe(v[r], v[r + 4]);
    }
};
template <typename E> struct rad<E, 16> {
    typedef typename scalar_of<E>::type T;
    static MM_HD void fwd(E* v)
    {
        const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, c = (T)0.70710678118654752440;
#pragma unroll
        for (int r = 0; r < 8; r++) bfe(v[r], v[r + 8]);
        // * w16^r = exp(-i pi r / 8)
        v[9] = crot(v[9], c1, -s1); v[10] = crot(v[10], c, -c); v[11] = crot(v[11], s1, -c1); v[12] = mul_mi(v[12]);
        v[13] = crot(v[13], -s1, -c1); v[14] = crot(v[14], -c, -c); v[15] = crot(v[15], -c1, -s1);
        rad<E, 8>::fwd(v); rad<E, 8>::fwd(v + 8);
    }
    static MM_HD void inv(E* v)
    {
        const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, c = (T)0.70710678118654752440;
        rad<E, 8>::inv(v); rad<E, 8>::inv(v + 8);
        v[9] = crot(v[9], c1, s1); v[10] = crot(v[10], c, c); v[11] = crot(v[11], s1, c1); v[12] = mul_pi(v[12]);
        v[13] = crot(v[13], -s1, c1); v[14] = crot(v[14], -c, c); v[15] = crot(v[15], -c1, s1);
#pragma unroll
        for (int r = 0; r < 8; r++) bfe(v[r], v[r + 8]);
    }
};
template <typename E> struct rad<E, 32> {
    typedef typename scalar_of<E>::type T;
    static MM_HD void tw32(int r, T& c, T& s)   // exp(-i pi r / 16), r = 1..15
    {
        const T C[16] = { (T)1.0, (T)0.98078528040323044913, (T)0.92387953251128675613, (T)0.83146961230254523708,
                          (T)0.70710678118654752440, (T)0.55557023301960222474, (T)0.38268343236508977173, (T)0.19509032201612826785,
                          (T)0.0, (T)-0.19509032201612826785, (T)-0.38268343236508977173, (T)-0.55557023301960222474,
                          (T)-0.70710678118654752440, (T)-0.83146961230254523708, (T)-0.92387953251128675613, (T)-0.98078528040323044913 };
        c = C[r]; s = -C[(r + 8) & 15] * (r < 8 ? (T)-1 : (T)1);
    }
    static MM_HD void fwd(E* v)
    {
#pragma unroll
        for (int r = 0; r < 16; r++) bfe(v[r], v[r + 16]);
#pragma unroll
        for (int r = 1; r < 16; r++) {
            T c, s; tw32(r, c, s);
            v[16 + r] = crot(v[16 + r], c, s);
        }
        rad<E, 16>::fwd(v); rad<E, 16>::fwd(v + 16);
    }
    static MM_HD void inv(E* v)
    {
        rad<E, 16>::inv(v); rad<E, 16>::inv(v + 16);
#pragma unroll
        for (int r = 1; r < 16; r++) {
            T c, s; tw32(r, c, s);
            v[16 + r] = crot(v[16 + r], c, -s);
        }
#pragma unroll
        for (int r = 0; r < 16; r++) bfe(v[r], v[r + 16]);
    }
};

// w0 * exp(-i pi r / R), r = 0..R-1: the pad / crop twiddles w_n^(i + r n/(2R)) of a pruned first / last
// stage derived from the single table value w0 = w_n^i (one load per butterfly instead of R)
template <typename T, int R> MM_HD void pad_twiddles(cx<T> w0, cx<T>* wp)
{
    const T c1 = (T)0.92387953251128675613, s1 = (T)0.38268343236508977173, c = (T)0.70710678118654752440;
    wp[0] = w0;
    if (R == 2) { wp[1] = mul_mi(w0); }
    else if (R == 4) { wp[1] = crot(w0, c, -c); wp[2] = mul_mi(w0); wp[3] = crot(w0, -c, -c); }
    else if (R == 8) {
        wp[1] = crot(w0, c1, -s1); wp[2] = crot(w0, c, -c); wp[3] = crot(w0, s1, -c1); wp[4] = mul_mi(w0);
        wp[5] = crot(w0, -s1, -c1); wp[6] = crot(w0, -c, -c); wp[7] = crot(w0, -c1, -s1);
    }
}

// a * w_n^k for compile-time n <= 64 and k < n/2 (the pad / crop twiddles of the register z transform): the twiddle is
// an immediate, not a table load.  w_64^j = cos(pi j / 32) - i sin(pi j / 32).
template <typename T> MM_HD void w64(int j, T& c, T& s)
{
    const T C[32] = { (T)1.00000000000000000000, (T)0.99518472667219692873, (T)0.98078528040323043058, (T)0.95694033573220882438, (T)0.92387953251128673848, (T)0.88192126434835504956, (T)0.83146961230254523567, (T)0.77301045336273699338, (T)0.70710678118654757274, (T)0.63439328416364548779, (T)0.55557023301960228867, (T)0.47139673682599780857, (T)0.38268343236508983729, (T)0.29028467725446233105, (T)0.19509032201612833135, (T)0.09801714032956077016, (T)0.00000000000000006123, (T)-0.09801714032956064526, (T)-0.19509032201612819257, (T)-0.29028467725446216452, (T)-0.38268343236508972627, (T)-0.47139673682599769755, (T)-0.55557023301960195560, (T)-0.63439328416364537677, (T)-0.70710678118654746172, (T)-0.77301045336273699338, (T)-0.83146961230254534669, (T)-0.88192126434835493853, (T)-0.92387953251128673848, (T)-0.95694033573220882438, (T)-0.98078528040323043058, (T)-0.99518472667219681771 };
    const T S[32] = { (T)0.00000000000000000000, (T)0.09801714032956060363, (T)0.19509032201612824808, (T)0.29028467725446233105, (T)0.38268343236508978178, (T)0.47139673682599764204, (T)0.55557023301960217765, (T)0.63439328416364548779, (T)0.70710678118654746172, (T)0.77301045336273699338, (T)0.83146961230254523567, (T)0.88192126434835493853, (T)0.92387953251128673848, (T)0.95694033573220893540, (T)0.98078528040323043058, (T)0.99518472667219681771, (T)1.00000000000000000000, (T)0.99518472667219692873, (T)0.98078528040323043058, (T)0.95694033573220893540, (T)0.92387953251128673848, (T)0.88192126434835504956, (T)0.83146961230254545772, (T)0.77301045336273710440, (T)0.70710678118654757274, (T)0.63439328416364548779, (T)0.55557023301960217765, (T)0.47139673682599786408, (T)0.38268343236508989280, (T)0.29028467725446238656, (T)0.19509032201612860891, (T)0.09801714032956082567 };
    c = C[j]; s = S[j];
}
template <typename T, int N> MM_HD cx<T> rot_w(cx<T> a, int k)      // a * w_N^k
{
    T c, s; w64<T>(k * (64 / N), c, s);
    return crot(a, c, -s);
}
template <typename T, int N> MM_HD cx<T> rot_wc(cx<T> a, int k)     // a * conj(w_N^k)
{
    T c, s; w64<T>(k * (64 / N), c, s);
    return crot(a, c, s);
}

// first radix of the v2 schedule for block length m >= 16: remainder first, then 8s
MM_HD int first_radix(int m) { int r = m; while (r > 8) r >>= 3; return r; }

}  // namespace mm
