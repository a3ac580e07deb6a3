/*
 * oracle/mo.c — the ORACLE: a plain, slow, obviously-correct CPU statement of the
 * micromagnetic LLG hot path of arxiv 2406.16064.
 *
 * THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may build, load or call it.  It shares no code,
 * header, table or helper with the CUDA library (paper_2406_16064_b200/csrc) and
 * neither includes the other.  All floating point is fp64, except the demagnetisation
 * tensor, which is evaluated in __float128 and rounded once (reading R1).
 *
 * What is stated here, and the passage each part follows:
 *   mo_newell_point / mo_newell_tensor  cell-averaged demag tensor N(r_i - r_j)
 *        PAPER.md:136 (§III.B, "demagnetization tensor ... 3x3 matrix [20]"); the closed
 *        forms f, g are those of ref [20], not printed in the paper —
 *        DESIGN.md reading R1.
 *   mo_demag_direct   H_d,i = - sum_j N_{i-j} M_j           PAPER.md:138 (Eq. 8), O(N^2)
 *   mo_demag_fft      the same sum as a zero-padded FFT convolution, 3 forward + 3
 *                     inverse transforms
 *   exchange          Eq. 5  PAPER.md:122       DMI  Eq. 15
 *   anisotropy        Eq. 32 PAPER.md:269 in its continuum reading (R6); cubic Eq. 33
 *   cell-based A, D   A_ij = 2 A_i A_j/(A_i + A_j) PAPER.md:120; D_ij likewise, D2d e_ij table
 *   Zeeman            Eq. 35
 *   LL right-hand side Eq. 37
 *   RK4 + projection  PAPER.md:425; Dormand-Prince + projection PAPER.md:298, ref [37]
 *   energy            Eq. 1, 2, 6/7, 10, 12 summed per cell
 *   mo_minimize       steepest descent with Barzilai-Borwein steps, Eq. 50-52
 *   Zhang-Li torque   f_stt of Eq. 44's text with tau = (u.grad) m, PAPER.md:306-308 (Eq. 38), :352; sign of u as in
 *                     Eq. 44 / Eq. 54 — Eq. 38 prints the opposite sign, R17
 *   Slonczewski / SOT Eq. 40, solved for dm/dt (LL form)
 *   thermal field     Eq. 41-42: one Gaussian vector per cell and step, held over the step's stages;
 *                     normals from Philox4x32-10 + Box-Muller keyed by (seed, step, cell) (R18)
 *   Cayley integrator Eq. 43-49: classical RK4 on omega (Eq. 49), restart (omega = 0) every step
 *
 * Layout: x fastest, idx = i + nx*(j + ny*k); vector fields are SoA, v[c*N + idx].
 * A neighbour is absent when outside the mesh or when its Ms is 0 (R4);
 * cells with Ms = 0 have H = 0, dm/dt = 0 and are left untouched (R5).
 *
 * Parity pins: tests/test_oracle_*.py (closed forms, printed worked values, brute
 * force).  The adaptive controller and relax end states are "parity unpinned" beyond
 * the step-by-step statement here (R8).
 */
#include <math.h>
#include <quadmath.h>
#include <stdlib.h>
#include <string.h>
#include <stdio.h>

#define MO_MU0 (4.0e-7 * 3.14159265358979323846264338327950288)

typedef __float128 qf;

typedef struct mo_sim {
    int nx, ny, nz;
    double dx, dy, dz;
    long N;
    double *Ms;                 /* N */
    double A, D, Ku, ux, uy, uz, hx, hy, hz, alpha, gamma;
    double Kc;                  /* cubic anisotropy constant (Eq. 33), crystal axes = mesh axes */
    double *Acell, *Dcell;      /* optional per-cell A_i, D_i (N each) or NULL: PAPER.md:120, 175 */
    double *Hcell;              /* optional per-cell external field (3N, SoA) or NULL: Eq. 35 with H_z,i */
    int dmi_kind;               /* 0 none, 1 bulk, 2 interfacial, 3 D2d */
    int integrator;             /* 0 RK4, 1 DOPRI5, 2 Cayley-transform RK4 (Eq. 49) */
    double stt_u[3], stt_beta;  /* Zhang-Li: u in m/s (Eq. 39), beta */
    int stt_on;
    double stt_b, stt_w;        /* time profile of the current: u(t) = u exp(-b t) cos(w t); 0, 0 = constant */
    double t_eval;              /* time at which the right-hand side is being evaluated (stage time inside a step) */
    int in_step;
    double sl_aJ, sl_bJ, sl_p[3]; /* Slonczewski / SOT (Eq. 40): a_J, b_J in 1/s, unit vector p */
    int sl_on;
    double temperature;         /* K; 0 = no thermal field */
    unsigned long long th_seed, th_step;   /* Philox key / number of step attempts so far */
    const double *Hth;          /* thermal field of the step in progress (3N) or NULL */
    int demag;                  /* 0 off, 1 FFT path, 2 direct O(N^2) sum */
    double *Nten;               /* 6 * N: xx,yy,zz,xy,xz,yz at offsets i>=0,j>=0,k>=0 */
    double *Khat;               /* 6 * P complex (interleaved) on the padded grid, or NULL */
    int px, py, pz;
    double t;
} mo_sim;

/* ------------------------------------------------------------------------------------
 * Demag tensor, ref [20] of the paper.  f is even in x, y, z;
 * g is odd in x, odd in y, even in z.  A term whose prefactor vanishes is 0.
 * ---------------------------------------------------------------------------------- */
static qf newell_f(qf x, qf y, qf z)
{
    x = fabsq(x); y = fabsq(y); z = fabsq(z);
    qf x2 = x * x, y2 = y * y, z2 = z * z;
    qf R = sqrtq(x2 + y2 + z2);
    qf r = 0;
    if (y > 0 && (x2 + z2) > 0) r += (y / 2) * (z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z > 0 && (x2 + y2) > 0) r += (z / 2) * (y2 - x2) * asinhq(z / sqrtq(x2 + y2));
    if (x > 0 && y > 0 && z > 0) r -= x * y * z * atanq(y * z / (x * R));
    r += (2 * x2 - y2 - z2) * R / 6;
    return r;
}

static qf newell_g(qf x, qf y, qf z)
{
    qf sign = 1;
    if (x < 0) sign = -sign;
    if (y < 0) sign = -sign;
    x = fabsq(x); y = fabsq(y); z = fabsq(z);
    qf x2 = x * x, y2 = y * y, z2 = z * z;
    qf R = sqrtq(x2 + y2 + z2);
    qf r = 0;
    if (x > 0 && y > 0 && z > 0) r += x * y * z * asinhq(z / sqrtq(x2 + y2));
    if (y > 0 && x > 0) r += (y / 6) * (3 * z2 - y2) * asinhq(x / sqrtq(y2 + z2));
    if (x > 0 && y > 0) r += (x / 6) * (3 * z2 - x2) * asinhq(y / sqrtq(x2 + z2));
    if (z > 0 && x > 0 && y > 0) {
        r -= (z * z2 / 6) * atanq(x * y / (z * R));
        r -= (z * y2 / 2) * atanq(x * z / (y * R));
        r -= (z * x2 / 2) * atanq(y * z / (x * R));
    }
    r -= x * y * R / 3;
    return sign * r;
}

/* N_xx(X,Y,Z) = 1/(4 pi V) sum_{p,q,r in {-1,0,1}} c_p c_q c_r f(X+p dx, Y+q dy, Z+r dz),
 * c_0 = 2, c_{+-1} = -1; N_xy the same with g. */
static qf newell_stencil(qf (*fn)(qf, qf, qf), qf X, qf Y, qf Z, qf dx, qf dy, qf dz)
{
    static const int c[3] = { -1, 2, -1 };
    qf s = 0;
    for (int p = -1; p <= 1; p++)
        for (int q = -1; q <= 1; q++)
            for (int r = -1; r <= 1; r++)
                s += (qf)(c[p + 1] * c[q + 1] * c[r + 1]) * fn(X + p * dx, Y + q * dy, Z + r * dz);
    return s / (4 * M_PIq * dx * dy * dz);
}

/* Six components at one displacement (X,Y,Z) [same length unit as dx,dy,dz].
 * Other components by permuting coordinates together with cell edges. out: xx,yy,zz,xy,xz,yz */
void mo_newell_point(double X, double Y, double Z, double dx, double dy, double dz, double out6[6])
{
    out6[0] = (double)newell_stencil(newell_f, X, Y, Z, dx, dy, dz);
    out6[1] = (double)newell_stencil(newell_f, Y, X, Z, dy, dx, dz);
    out6[2] = (double)newell_stencil(newell_f, Z, Y, X, dz, dy, dx);
    out6[3] = (double)newell_stencil(newell_g, X, Y, Z, dx, dy, dz);
    out6[4] = (double)newell_stencil(newell_g, X, Z, Y, dx, dz, dy);
    out6[5] = (double)newell_stencil(newell_g, Y, Z, X, dy, dz, dx);
}

/* Tensor at all offsets (i,j,k), 0<=i<nx, 0<=j<ny, 0<=k<nz.  f and g are evaluated once
 * per lattice point (they are shared between neighbouring stencils) — the same sum as
 * newell_stencil, only with the function values tabulated. out[c*N + i + nx*(j + ny*k)]. */
void mo_newell_tensor(int nx, int ny, int nz, double dx, double dy, double dz, double *out)
{
    const long N = (long)nx * ny * nz;
    const int gx = nx + 1, gy = ny + 1, gz = nz + 1;      /* lattice points 0..n (|-1| = 1) */
    const long G = (long)gx * gy * gz;
    qf *tab = (qf *)malloc(sizeof(qf) * G);
    static const int c[3] = { -1, 2, -1 };
    const qf pref = 1 / (4 * M_PIq * (qf)dx * (qf)dy * (qf)dz);
    for (int comp = 0; comp < 6; comp++) {
#pragma omp parallel for collapse(2) schedule(dynamic, 4)
        for (int k = 0; k < gz; k++)
            for (int j = 0; j < gy; j++)
                for (int i = 0; i < gx; i++) {
                    qf x = i * (qf)dx, y = j * (qf)dy, z = k * (qf)dz, v;
                    switch (comp) {
                    case 0: v = newell_f(x, y, z); break;
                    case 1: v = newell_f(y, x, z); break;
                    case 2: v = newell_f(z, y, x); break;
                    case 3: v = newell_g(x, y, z); break;
                    case 4: v = newell_g(x, z, y); break;
                    default: v = newell_g(y, z, x); break;
                    }
                    tab[i + (long)gx * (j + (long)gy * k)] = v;
                }
        /* which two axes the tabulated function is odd in (none for the diagonal) */
        const int oddx = (comp == 3 || comp == 4), oddy = (comp == 3 || comp == 5), oddz = (comp == 4 || comp == 5);
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < nz; k++)
            for (int j = 0; j < ny; j++)
                for (int i = 0; i < nx; i++) {
                    qf s = 0;
                    for (int p = -1; p <= 1; p++)
                        for (int q = -1; q <= 1; q++)
                            for (int r = -1; r <= 1; r++) {
                                int a = i + p, b = j + q, cc = k + r, sg = 1;
                                if (a < 0) { a = -a; if (oddx) sg = -sg; }
                                if (b < 0) { b = -b; if (oddy) sg = -sg; }
                                if (cc < 0) { cc = -cc; if (oddz) sg = -sg; }
                                s += (qf)(sg * c[p + 1] * c[q + 1] * c[r + 1]) * tab[a + (long)gx * (b + (long)gy * cc)];
                            }
                    out[comp * N + i + (long)nx * (j + (long)ny * k)] = (double)(s * pref);
                }
    }
    free(tab);
}

/* N_ab at a signed offset from the non-negative-octant table: diagonal components are even
 * in every axis, N_ab (a != b) is odd in axes a and b (symmetric, depends on
 * r_i - r_j only). */
static inline void tensor_at(const mo_sim *s, int di, int dj, int dk, double n[6])
{
    int sx = di < 0 ? -1 : 1, sy = dj < 0 ? -1 : 1, sz = dk < 0 ? -1 : 1;
    long o = abs(di) + (long)s->nx * (abs(dj) + (long)s->ny * abs(dk));
    n[0] = s->Nten[0 * s->N + o];
    n[1] = s->Nten[1 * s->N + o];
    n[2] = s->Nten[2 * s->N + o];
    n[3] = s->Nten[3 * s->N + o] * (sx * sy);
    n[4] = s->Nten[4 * s->N + o] * (sx * sz);
    n[5] = s->Nten[5 * s->N + o] * (sy * sz);
}

/* ------------------------------------------------------------------------------------
 * Eq. 8 written out: H_d,i = - sum_j N_{i-j} (Ms_j m_j), all pairs.
 * ---------------------------------------------------------------------------------- */
static void demag_direct(const mo_sim *s, const double *m, double *H)
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const long N = s->N;
#pragma omp parallel for schedule(static)
    for (long i = 0; i < N; i++) {
        int ix = (int)(i % nx), iy = (int)((i / nx) % ny), iz = (int)(i / ((long)nx * ny));
        double hx = 0, hy = 0, hz = 0;
        for (int kz = 0; kz < nz; kz++)
            for (int ky = 0; ky < ny; ky++)
                for (int kx = 0; kx < nx; kx++) {
                    long j = kx + (long)nx * (ky + (long)ny * kz);
                    double Msj = s->Ms[j];
                    if (Msj == 0.0) continue;
                    double n[6];
                    tensor_at(s, ix - kx, iy - ky, iz - kz, n);
                    double Mx = Msj * m[j], My = Msj * m[N + j], Mz = Msj * m[2 * N + j];
                    hx -= n[0] * Mx + n[3] * My + n[4] * Mz;
                    hy -= n[3] * Mx + n[1] * My + n[5] * Mz;
                    hz -= n[4] * Mx + n[5] * My + n[2] * Mz;
                }
        H[i] = hx; H[N + i] = hy; H[2 * N + i] = hz;
    }
}

/* One sampled output of Eq. 8 (used for full-size parity on sampled cells). */
void mo_demag_direct_at(const mo_sim *s, const double *m, long cell, double h3[3])
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const long N = s->N;
    int ix = (int)(cell % nx), iy = (int)((cell / nx) % ny), iz = (int)(cell / ((long)nx * ny));
    double hx = 0, hy = 0, hz = 0;
#pragma omp parallel for collapse(2) reduction(+ : hx, hy, hz) schedule(static)
    for (int kz = 0; kz < nz; kz++)
        for (int ky = 0; ky < ny; ky++)
            for (int kx = 0; kx < nx; kx++) {
                long j = kx + (long)nx * (ky + (long)ny * kz);
                double Msj = s->Ms[j];
                if (Msj == 0.0) continue;
                double n[6];
                tensor_at(s, ix - kx, iy - ky, iz - kz, n);
                double Mx = Msj * m[j], My = Msj * m[N + j], Mz = Msj * m[2 * N + j];
                hx -= n[0] * Mx + n[3] * My + n[4] * Mz;
                hy -= n[3] * Mx + n[1] * My + n[5] * Mz;
                hz -= n[4] * Mx + n[5] * My + n[2] * Mz;
            }
    h3[0] = hx; h3[1] = hy; h3[2] = hz;
}

/* ------------------------------------------------------------------------------------
 * Own FFT: textbook recursive radix-2 decimation in time, complex fp64, interleaved.
 * sign = -1 forward, +1 inverse (unscaled).
 * ---------------------------------------------------------------------------------- */
static void fft_rec(double *a, double *tmp, int n, int sign)
{
    if (n == 1) return;
    int h = n / 2;
    for (int i = 0; i < h; i++) {
        tmp[2 * i] = a[4 * i];         tmp[2 * i + 1] = a[4 * i + 1];           /* even */
        tmp[2 * (h + i)] = a[4 * i + 2]; tmp[2 * (h + i) + 1] = a[4 * i + 3];   /* odd  */
    }
    memcpy(a, tmp, sizeof(double) * 2 * n);
    fft_rec(a, tmp, h, sign);
    fft_rec(a + 2 * h, tmp, h, sign);
    for (int k = 0; k < h; k++) {
        double ang = sign * 2.0 * M_PI * (double)k / (double)n;
        double wr = cos(ang), wi = sin(ang);
        double er = a[2 * k], ei = a[2 * k + 1];
        double orr = a[2 * (h + k)], oi = a[2 * (h + k) + 1];
        double tr = wr * orr - wi * oi, ti = wr * oi + wi * orr;
        a[2 * k] = er + tr;       a[2 * k + 1] = ei + ti;
        a[2 * (h + k)] = er - tr; a[2 * (h + k) + 1] = ei - ti;
    }
}

/* 1-D transform of every line along `axis` of a px*py*pz complex array */
static void fft3d_axis(double *a, int px, int py, int pz, int axis, int sign)
{
    int n = axis == 0 ? px : axis == 1 ? py : pz;
    if (n == 1) return;
    long stride = axis == 0 ? 1 : axis == 1 ? px : (long)px * py;
    long nlines = (long)px * py * pz / n;
#pragma omp parallel
    {
        double *line = (double *)malloc(sizeof(double) * 2 * n);
        double *tmp = (double *)malloc(sizeof(double) * 2 * n);
#pragma omp for schedule(static)
        for (long l = 0; l < nlines; l++) {
            long base;
            if (axis == 0) base = l * px;
            else if (axis == 1) base = (l % px) + (l / px) * (long)px * py;
            else base = l;
            for (int i = 0; i < n; i++) {
                line[2 * i] = a[2 * (base + i * stride)];
                line[2 * i + 1] = a[2 * (base + i * stride) + 1];
            }
            fft_rec(line, tmp, n, sign);
            for (int i = 0; i < n; i++) {
                a[2 * (base + i * stride)] = line[2 * i];
                a[2 * (base + i * stride) + 1] = line[2 * i + 1];
            }
        }
        free(line); free(tmp);
    }
}

static void fft3d(double *a, int px, int py, int pz, int sign)
{
    fft3d_axis(a, px, py, pz, 0, sign);
    fft3d_axis(a, px, py, pz, 1, sign);
    fft3d_axis(a, px, py, pz, 2, sign);
}

/* Kernel array on the padded grid with wrap indexing (R3):
 * padded index p is offset p for p<n, p-2n for p>n, the slot p=n is 0; axes with n=1 are
 * not padded.  Khat = FFT of it. */
static void build_khat(mo_sim *s)
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const int px = s->px, py = s->py, pz = s->pz;
    const long P = (long)px * py * pz;
    s->Khat = (double *)calloc((size_t)12 * P, sizeof(double));
    for (int c = 0; c < 6; c++) {
        double *K = s->Khat + (size_t)2 * P * c;
#pragma omp parallel for collapse(2) schedule(static)
        for (int c3 = 0; c3 < pz; c3++)
            for (int b = 0; b < py; b++)
                for (int a = 0; a < px; a++) {
                    if ((nx > 1 && a == nx) || (ny > 1 && b == ny) || (nz > 1 && c3 == nz)) continue;
                    int di = a < nx ? a : a - px, dj = b < ny ? b : b - py, dk = c3 < nz ? c3 : c3 - pz;
                    double n[6];
                    tensor_at(s, di, dj, dk, n);
                    K[2 * (a + (long)px * (b + (long)py * c3))] = n[c];
                }
        fft3d(K, px, py, pz, -1);
    }
}

/* H_d = crop( IFFT( - Khat . FFT( pad(Ms m) ) ) ) */
static void demag_fft(mo_sim *s, const double *m, double *H)
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const int px = s->px, py = s->py, pz = s->pz;
    const long P = (long)px * py * pz, N = s->N;
    if (!s->Khat) build_khat(s);
    double *M = (double *)calloc((size_t)6 * P, sizeof(double));
    double *Hk = (double *)calloc((size_t)6 * P, sizeof(double));
    for (int c = 0; c < 3; c++) {
        double *Mc = M + (size_t)2 * P * c;
        for (int k = 0; k < nz; k++)
            for (int j = 0; j < ny; j++)
                for (int i = 0; i < nx; i++) {
                    long q = i + (long)nx * (j + (long)ny * k);
                    Mc[2 * (i + (long)px * (j + (long)py * k))] = s->Ms[q] * m[c * N + q];
                }
        fft3d(Mc, px, py, pz, -1);
    }
    const double *K = s->Khat;
    /* row a of the symmetric tensor uses components: x:(xx,xy,xz) y:(xy,yy,yz) z:(xz,yz,zz) */
    static const int row[3][3] = { { 0, 3, 4 }, { 3, 1, 5 }, { 4, 5, 2 } };
    for (int a = 0; a < 3; a++) {
        double *Ha = Hk + (size_t)2 * P * a;
#pragma omp parallel for schedule(static)
        for (long q = 0; q < P; q++) {
            double re = 0, im = 0;
            for (int b = 0; b < 3; b++) {
                const double *Kc = K + (size_t)2 * P * row[a][b];
                const double *Mb = M + (size_t)2 * P * b;
                re += Kc[2 * q] * Mb[2 * q] - Kc[2 * q + 1] * Mb[2 * q + 1];
                im += Kc[2 * q] * Mb[2 * q + 1] + Kc[2 * q + 1] * Mb[2 * q];
            }
            Ha[2 * q] = -re; Ha[2 * q + 1] = -im;
        }
        fft3d(Ha, px, py, pz, +1);
        for (int k = 0; k < nz; k++)
            for (int j = 0; j < ny; j++)
                for (int i = 0; i < nx; i++)
                    H[a * N + i + (long)nx * (j + (long)ny * k)] = Ha[2 * (i + (long)px * (j + (long)py * k))] / (double)P;
    }
    free(M); free(Hk);
}

/* ------------------------------------------------------------------------------------
 * Local terms.  which: bit0 exchange, bit1 DMI, bit2 uniaxial anisotropy, bit3 Zeeman, bit5 cubic anisotropy.  Adds to H.
 * ---------------------------------------------------------------------------------- */
static void local_field_add(const mo_sim *s, const double *m, double *H, int which)
{
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const long N = s->N;
    const double un = sqrt(s->ux * s->ux + s->uy * s->uy + s->uz * s->uz);
    const double ux = un > 0 ? s->ux / un : 0, uy = un > 0 ? s->uy / un : 0, uz = un > 0 ? s->uz / un : 0;
    /* neighbour order: -x, +x, -y, +y, -z, +z */
    static const int off[6][3] = { { -1, 0, 0 }, { 1, 0, 0 }, { 0, -1, 0 }, { 0, 1, 0 }, { 0, 0, -1 }, { 0, 0, 1 } };
    /* DMI vectors e_ij: bulk r^_ij; interfacial e_z x r^_ij; D2d {e_x,-e_x,-e_y,e_y,0,0} */
    static const double e_bulk[6][3] = { { -1, 0, 0 }, { 1, 0, 0 }, { 0, -1, 0 }, { 0, 1, 0 }, { 0, 0, -1 }, { 0, 0, 1 } };
    static const double e_int[6][3] = { { 0, -1, 0 }, { 0, 1, 0 }, { 1, 0, 0 }, { -1, 0, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
    static const double e_d2d[6][3] = { { 1, 0, 0 }, { -1, 0, 0 }, { 0, -1, 0 }, { 0, 1, 0 }, { 0, 0, 0 }, { 0, 0, 0 } };
    const double delta[6] = { s->dx, s->dx, s->dy, s->dy, s->dz, s->dz };
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                long q = i + (long)nx * (j + (long)ny * k);
                double Msi = s->Ms[q];
                if (Msi == 0.0) continue;
                double mx = m[q], my = m[N + q], mz = m[2 * N + q];
                double hx = 0, hy = 0, hz = 0;
                for (int nb = 0; nb < 6; nb++) {
                    int a = i + off[nb][0], b = j + off[nb][1], c = k + off[nb][2];
                    if (a < 0 || a >= nx || b < 0 || b >= ny || c < 0 || c >= nz) continue;
                    long p = a + (long)nx * (b + (long)ny * c);
                    if (s->Ms[p] == 0.0) continue;
                    double nxm = m[p], nym = m[N + p], nzm = m[2 * N + p];
                    if (which & 1) {           /* Eq. 5; A_ij = A, or 2 A_i A_j / (A_i + A_j) for cell-based A */
                        double Aij = s->A;
                        if (s->Acell) {
                            const double Ai = s->Acell[q], Aj = s->Acell[p];
                            Aij = (Ai + Aj) != 0.0 ? 2.0 * Ai * Aj / (Ai + Aj) : 0.0;
                        }
                        double f = 2.0 * Aij / (MO_MU0 * Msi) / (delta[nb] * delta[nb]);
                        hx += f * (nxm - mx); hy += f * (nym - my); hz += f * (nzm - mz);
                    }
                    if ((which & 2) && s->dmi_kind != 0) {   /* Eq. 15; D_ij = D, or 2 D_i D_j / (D_i + D_j) */
                        const double *e = s->dmi_kind == 1 ? e_bulk[nb] : (s->dmi_kind == 2 ? e_int[nb] : e_d2d[nb]);
                        double Dij = s->D;
                        if (s->Dcell) {
                            const double Di = s->Dcell[q], Dj = s->Dcell[p];
                            Dij = (Di + Dj) != 0.0 ? 2.0 * Di * Dj / (Di + Dj) : 0.0;
                        }
                        double f = -Dij / (MO_MU0 * Msi) / delta[nb];
                        hx += f * (e[1] * nzm - e[2] * nym);
                        hy += f * (e[2] * nxm - e[0] * nzm);
                        hz += f * (e[0] * nym - e[1] * nxm);
                    }
                }
                if (which & 4) {               /* 2Ku/(mu0 Ms) (m.u) u */
                    double f = 2.0 * s->Ku / (MO_MU0 * Msi) * (mx * ux + my * uy + mz * uz);
                    hx += f * ux; hy += f * uy; hz += f * uz;
                }
                if (which & 32) {              /* cubic anisotropy, Eq. 33 w = Kc (mx^4 + my^4 + mz^4) in its continuum
                                                * reading (R6): H = -(1/(mu0 Ms)) dw/dm = -(4 Kc/(mu0 Ms)) (mx^3, my^3, mz^3) */
                    double f = -4.0 * s->Kc / (MO_MU0 * Msi);
                    hx += f * mx * mx * mx; hy += f * my * my * my; hz += f * mz * mz * mz;
                }
                if (which & 8) {               /* Eq. 35: the external field itself, uniform or per cell */
                    if (s->Hcell) { hx += s->Hcell[q]; hy += s->Hcell[N + q]; hz += s->Hcell[2 * N + q]; }
                    else { hx += s->hx; hy += s->hy; hz += s->hz; }
                }
                H[q] += hx; H[N + q] += hy; H[2 * N + q] += hz;
            }
}

/* which: bits 0..3 and 5 as above, bit4 demag */
int mo_field_terms(mo_sim *s, const double *m, double *H, int which)
{
    const long N = s->N;
    memset(H, 0, sizeof(double) * 3 * N);
    if ((which & 16) && s->demag) {
        if (!s->Nten) return -3;
        /* the own FFT is radix-2: meshes whose padded sizes are not powers of two take the defining direct sum */
        const int pow2 = !(s->px & (s->px - 1)) && !(s->py & (s->py - 1)) && !(s->pz & (s->pz - 1));
        if (s->demag == 2 || !pow2) demag_direct(s, m, H); else demag_fft(s, m, H);
        for (long q = 0; q < N; q++)
            if (s->Ms[q] == 0.0) H[q] = H[N + q] = H[2 * N + q] = 0.0;
    }
    local_field_add(s, m, H, which & (15 | 32));
    return 0;
}

int mo_effective_field(mo_sim *s, const double *m, double *H) { return mo_field_terms(s, m, H, 63); }

/* ------------------------------------------------------------------------------------
 * Counter-based normals for the thermal field (R18): Philox4x32-10 (Salmon et al., SC'11: 10 rounds of
 * two 32x32->64 multiplies with the constants below, key bumped by the Weyl constants between rounds) on
 * counter = (cell lo, cell hi, step lo, step hi), key = (seed lo, seed hi); four 32-bit words x -> u = (x + 1/2) 2^-32
 * in (0, 1); Box-Muller: (u0, u1) -> sqrt(-2 ln u0) (cos, sin)(2 pi u1) = (eta_x, eta_y), (u2, u3) -> eta_z (the sine
 * of the second pair is not used).
 * ---------------------------------------------------------------------------------- */
void mo_philox4x32_10(const unsigned int ctr[4], const unsigned int key[2], unsigned int out[4])
{
    unsigned int c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
    for (int r = 0; r < 10; r++) {
        unsigned long long p0 = (unsigned long long)0xD2511F53u * c0, p1 = (unsigned long long)0xCD9E8D57u * c2;
        unsigned int n0 = (unsigned int)(p1 >> 32) ^ c1 ^ k0, n1 = (unsigned int)p1;
        unsigned int n2 = (unsigned int)(p0 >> 32) ^ c3 ^ k1, n3 = (unsigned int)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

void mo_normals3(unsigned long long seed, unsigned long long step, unsigned long long cell, double eta[3])
{
    const unsigned int ctr[4] = { (unsigned int)cell, (unsigned int)(cell >> 32), (unsigned int)step, (unsigned int)(step >> 32) };
    const unsigned int key[2] = { (unsigned int)seed, (unsigned int)(seed >> 32) };
    unsigned int x[4];
    mo_philox4x32_10(ctr, key, x);
    const double two_pi = 6.283185307179586476925286766559;
    double u[4];
    for (int i = 0; i < 4; i++) u[i] = ((double)x[i] + 0.5) * (1.0 / 4294967296.0);
    const double r0 = sqrt(-2.0 * log(u[0])), r1 = sqrt(-2.0 * log(u[2]));
    eta[0] = r0 * cos(two_pi * u[1]);
    eta[1] = r0 * sin(two_pi * u[1]);
    eta[2] = r1 * cos(two_pi * u[3]);
}

#define MO_KB 1.380649e-23

/* Eq. 42: xi_i^u = eta sqrt(2 alpha kB T / (mu0 Ms_i gamma V dt)), V = cell volume; 0 where Ms = 0 */
int mo_thermal_field(const mo_sim *s, double dt, unsigned long long step, double *xi)
{
    const long N = s->N;
    const double V = s->dx * s->dy * s->dz;
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0 || !(s->temperature > 0.0)) { xi[q] = xi[N + q] = xi[2 * N + q] = 0.0; continue; }
        double eta[3];
        mo_normals3(s->th_seed, step, (unsigned long long)q, eta);
        const double amp = sqrt(2.0 * s->alpha * MO_KB * s->temperature / (MO_MU0 * s->Ms[q] * s->gamma * V * dt));
        for (int c = 0; c < 3; c++) xi[c * N + q] = eta[c] * amp;
    }
    return 0;
}

/* tau = (u . grad) m by central differences, tau_i = sum_a u_a (m_{i+a} - m_{i-a}) / (2 Delta_a); an absent
 * neighbour (outside the mesh or Ms = 0) is replaced by the cell's own m (zero normal derivative, the free boundary
 * of R4; the paper prints no discretisation: DESIGN.md R17) */
int mo_stt_tau(mo_sim *s, const double *m, double *tau)
{
    if (!s->in_step) s->t_eval = s->t;
    const int nx = s->nx, ny = s->ny, nz = s->nz;
    const long N = s->N;
    const double delta[3] = { s->dx, s->dy, s->dz };
    for (int k = 0; k < nz; k++)
        for (int j = 0; j < ny; j++)
            for (int i = 0; i < nx; i++) {
                long q = i + (long)nx * (j + (long)ny * k);
                tau[q] = tau[N + q] = tau[2 * N + q] = 0.0;
                if (s->Ms[q] == 0.0) continue;
                const int pos[3] = { i, j, k }, lim[3] = { nx, ny, nz };
                const long str[3] = { 1, nx, (long)nx * ny };
                for (int a = 0; a < 3; a++) {
                    long pm = q, pp = q;
                    if (pos[a] > 0 && s->Ms[q - str[a]] != 0.0) pm = q - str[a];
                    if (pos[a] < lim[a] - 1 && s->Ms[q + str[a]] != 0.0) pp = q + str[a];
                    for (int c = 0; c < 3; c++) tau[c * N + q] += s->stt_u[a] * (m[c * N + pp] - m[c * N + pm]) / (2.0 * delta[a]);
                }
                /* u(t) = u exp(-b t) cos(w t) at the evaluation time ("u(t) = u0 e^{-bt} cos(wt)") */
                if (s->stt_b != 0.0 || s->stt_w != 0.0) {
                    const double f = exp(-s->stt_b * s->t_eval) * cos(s->stt_w * s->t_eval);
                    for (int c = 0; c < 3; c++) tau[c * N + q] *= f;
                }
            }
    return 0;
}

static void cross3(const double a[3], const double b[3], double c[3])
{
    c[0] = a[1] * b[2] - a[2] * b[1]; c[1] = a[2] * b[0] - a[0] * b[2]; c[2] = a[0] * b[1] - a[1] * b[0];
}

/* Eq. 37 with the thermal field of the step in progress added to H_eff, plus
 *  - Zhang-Li: dm/dt += f_stt x m, f_stt = [(beta - alpha) tau + (1 + alpha beta) m x tau]/(1 + alpha^2)
 *  - Slonczewski / SOT, Eq. 40: with T = -a_J m x (m x p) - b_J m x p the implicit equation
 *    dm/dt = ... + alpha m x dm/dt + T solves to dm/dt += (T + alpha m x T)/(1 + alpha^2). */
int mo_llg_rhs(mo_sim *s, const double *m, double *dmdt)
{
    const long N = s->N;
    if (!s->in_step) s->t_eval = s->t;
    double *H = (double *)malloc(sizeof(double) * 3 * N);
    int rc = mo_effective_field(s, m, H);
    if (rc) { free(H); return rc; }
    if (s->Hth) for (long q = 0; q < 3 * N; q++) H[q] += s->Hth[q];
    double *tau = NULL;
    if (s->stt_on) { tau = (double *)malloc(sizeof(double) * 3 * N); mo_stt_tau(s, m, tau); }
    const double gp = s->gamma / (1.0 + s->alpha * s->alpha), al = s->alpha;
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) { dmdt[q] = dmdt[N + q] = dmdt[2 * N + q] = 0.0; continue; }
        double mx = m[q], my = m[N + q], mz = m[2 * N + q];
        double hx = H[q], hy = H[N + q], hz = H[2 * N + q];
        double ax = my * hz - mz * hy, ay = mz * hx - mx * hz, az = mx * hy - my * hx;   /* m x H */
        double bx = my * az - mz * ay, by = mz * ax - mx * az, bz = mx * ay - my * ax;   /* m x (m x H) */
        dmdt[q] = -gp * ax - al * gp * bx;
        dmdt[N + q] = -gp * ay - al * gp * by;
        dmdt[2 * N + q] = -gp * az - al * gp * bz;
        const double mv[3] = { mx, my, mz };
        if (s->stt_on) {
            const double t[3] = { tau[q], tau[N + q], tau[2 * N + q] };
            double mt[3], f[3], fm[3];
            cross3(mv, t, mt);
            for (int c = 0; c < 3; c++) f[c] = ((s->stt_beta - al) * t[c] + (1.0 + al * s->stt_beta) * mt[c]) / (1.0 + al * al);
            cross3(f, mv, fm);
            for (int c = 0; c < 3; c++) dmdt[c * N + q] += fm[c];
        }
        if (s->sl_on) {
            double mp[3], mmp[3], T[3], mT[3];
            cross3(mv, s->sl_p, mp);
            cross3(mv, mp, mmp);
            for (int c = 0; c < 3; c++) T[c] = -s->sl_aJ * mmp[c] - s->sl_bJ * mp[c];
            cross3(mv, T, mT);
            for (int c = 0; c < 3; c++) dmdt[c * N + q] += (T[c] + al * mT[c]) / (1.0 + al * al);
        }
    }
    free(H); free(tau);
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Cayley transform.  Eq. 47: Q = (I - Omega/2)^-1 (I + Omega/2), Omega = skew[omega] (Eq. 45);
 * m = Q m0 (Eq. 43) by solving (I - Omega/2) x = (I + Omega/2) m0 with Cramer's rule.
 * ---------------------------------------------------------------------------------- */
void mo_cayley_apply(const double w[3], const double m0[3], double out[3])
{
    /* skew[w] = [[0,-w3,w2],[w3,0,-w1],[-w2,w1,0]] */
    const double h[3] = { 0.5 * w[0], 0.5 * w[1], 0.5 * w[2] };
    const double B[3][3] = { { 1, h[2], -h[1] }, { -h[2], 1, h[0] }, { h[1], -h[0], 1 } };      /* I - Omega/2 */
    const double C[3][3] = { { 1, -h[2], h[1] }, { h[2], 1, -h[0] }, { -h[1], h[0], 1 } };      /* I + Omega/2 */
    double r[3];
    for (int i = 0; i < 3; i++) r[i] = C[i][0] * m0[0] + C[i][1] * m0[1] + C[i][2] * m0[2];
    const double det = B[0][0] * (B[1][1] * B[2][2] - B[1][2] * B[2][1]) - B[0][1] * (B[1][0] * B[2][2] - B[1][2] * B[2][0])
                     + B[0][2] * (B[1][0] * B[2][1] - B[1][1] * B[2][0]);
    for (int c = 0; c < 3; c++) {
        double M[3][3];
        for (int i = 0; i < 3; i++) for (int j = 0; j < 3; j++) M[i][j] = j == c ? r[i] : B[i][j];
        out[c] = (M[0][0] * (M[1][1] * M[2][2] - M[1][2] * M[2][1]) - M[0][1] * (M[1][0] * M[2][2] - M[1][2] * M[2][0])
                  + M[0][2] * (M[1][0] * M[2][1] - M[1][1] * M[2][0])) / det;
    }
}

/* f of Eq. 44 at the magnetisation mm: gamma (H + alpha m x H)/(1 + alpha^2) with H = H_eff (+ thermal field of the
 * step) (+ the Slonczewski terms written as a field, (a_J/gamma) m x p + (b_J/gamma) p: "can be
 * incorporated into the effective fields"), plus f_stt. */
static int cayley_f(mo_sim *s, const double *mm, double *f)
{
    const long N = s->N;
    double *H = (double *)malloc(sizeof(double) * 3 * N);
    int rc = mo_effective_field(s, mm, H);
    if (rc) { free(H); return rc; }
    if (s->Hth) for (long q = 0; q < 3 * N; q++) H[q] += s->Hth[q];
    double *tau = NULL;
    if (s->stt_on) { tau = (double *)malloc(sizeof(double) * 3 * N); mo_stt_tau(s, mm, tau); }
    const double al = s->alpha, den = 1.0 + al * al;
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) { f[q] = f[N + q] = f[2 * N + q] = 0.0; continue; }
        const double mv[3] = { mm[q], mm[N + q], mm[2 * N + q] };
        double Hv[3] = { H[q], H[N + q], H[2 * N + q] }, mH[3];
        if (s->sl_on) {
            double mp[3];
            cross3(mv, s->sl_p, mp);
            for (int c = 0; c < 3; c++) Hv[c] += (s->sl_aJ * mp[c] + s->sl_bJ * s->sl_p[c]) / s->gamma;
        }
        cross3(mv, Hv, mH);
        for (int c = 0; c < 3; c++) f[c * N + q] = s->gamma * (Hv[c] + al * mH[c]) / den;
        if (s->stt_on) {
            const double t[3] = { tau[q], tau[N + q], tau[2 * N + q] };
            double mt[3];
            cross3(mv, t, mt);
            for (int c = 0; c < 3; c++) f[c * N + q] += ((s->stt_beta - al) * t[c] + (1.0 + al * s->stt_beta) * mt[c]) / den;
        }
    }
    free(H); free(tau);
    return 0;
}

/* d omega/dt of Eq. 49 at omega, for the step that started at m0: m = Q(omega) m0 (Eq. 43, 47), f = f(m) */
static int cayley_rhs(mo_sim *s, const double *m0, const double *w, double *mm, double *f, double *dw)
{
    const long N = s->N;
    for (long q = 0; q < N; q++) {
        const double wv[3] = { w[q], w[N + q], w[2 * N + q] }, m0v[3] = { m0[q], m0[N + q], m0[2 * N + q] };
        double o[3];
        mo_cayley_apply(wv, m0v, o);
        for (int c = 0; c < 3; c++) mm[c * N + q] = s->Ms[q] == 0.0 ? m0v[c] : o[c];
    }
    int rc = cayley_f(s, mm, f);
    if (rc) return rc;
    for (long q = 0; q < N; q++) {
        const double wv[3] = { w[q], w[N + q], w[2 * N + q] }, fv[3] = { f[q], f[N + q], f[2 * N + q] };
        double wf[3];
        cross3(wv, fv, wf);
        const double d = wv[0] * fv[0] + wv[1] * fv[1] + wv[2] * fv[2];
        for (int c = 0; c < 3; c++) dw[c * N + q] = fv[c] - 0.5 * wf[c] + 0.25 * d * wv[c];
    }
    return 0;
}

/* One step of the Cayley-transform integrator: omega(0) = 0 (restart every step), classical RK4 on
 * Eq. 49 over dt, m <- Q(omega(dt)) m.  No projection is applied: Q is a rotation.  max|dm/dt| = max_i |f_1 x m|. */
static int cayley_step(mo_sim *s, double *m, double dt, double *max_dmdt)
{
    const long N = s->N, n3 = 3 * N;
    double *k = (double *)malloc(sizeof(double) * n3 * 4), *w = (double *)calloc(n3, sizeof(double));
    double *mm = (double *)malloc(sizeof(double) * n3), *f = (double *)malloc(sizeof(double) * n3);
    int rc;
    s->t_eval = s->t;
    if ((rc = cayley_rhs(s, m, w, mm, f, k))) goto done;
    if (max_dmdt) {
        double mx = 0;
        for (long q = 0; q < N; q++) {
            if (s->Ms[q] == 0.0) continue;
            const double fv[3] = { f[q], f[N + q], f[2 * N + q] }, mv[3] = { m[q], m[N + q], m[2 * N + q] };
            double c[3];
            cross3(fv, mv, c);
            const double n = sqrt(c[0] * c[0] + c[1] * c[1] + c[2] * c[2]);
            if (n > mx || n != n) mx = n;
        }
        *max_dmdt = mx;
    }
    for (long q = 0; q < n3; q++) w[q] = 0.5 * dt * k[q];
    s->t_eval = s->t + 0.5 * dt;
    if ((rc = cayley_rhs(s, m, w, mm, f, k + n3))) goto done;
    for (long q = 0; q < n3; q++) w[q] = 0.5 * dt * k[n3 + q];
    if ((rc = cayley_rhs(s, m, w, mm, f, k + 2 * n3))) goto done;
    for (long q = 0; q < n3; q++) w[q] = dt * k[2 * n3 + q];
    s->t_eval = s->t + dt;
    if ((rc = cayley_rhs(s, m, w, mm, f, k + 3 * n3))) goto done;
    for (long q = 0; q < n3; q++) w[q] = dt / 6.0 * (k[q] + 2 * k[n3 + q] + 2 * k[2 * n3 + q] + k[3 * n3 + q]);
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) continue;
        const double wv[3] = { w[q], w[N + q], w[2 * N + q] }, m0v[3] = { m[q], m[N + q], m[2 * N + q] };
        double o[3];
        mo_cayley_apply(wv, m0v, o);
        for (int c = 0; c < 3; c++) m[c * N + q] = o[c];
    }
    s->t += dt;
done:
    free(k); free(w); free(mm); free(f);
    return rc;
}

static void project(const mo_sim *s, double *m)
{
    const long N = s->N;
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) continue;
        double n = sqrt(m[q] * m[q] + m[N + q] * m[N + q] + m[2 * N + q] * m[2 * N + q]);
        m[q] /= n; m[N + q] /= n; m[2 * N + q] /= n;
    }
}

static double max_norm(const mo_sim *s, const double *v)
{
    const long N = s->N;
    double mx = 0;
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) continue;
        double n = sqrt(v[q] * v[q] + v[N + q] * v[N + q] + v[2 * N + q] * v[2 * N + q]);
        if (n > mx || n != n) mx = n;
    }
    return mx;
}

/* Dormand-Prince 5(4) tableau, ref [37] of the paper; R8 */
static const double DP_A[7][6] = {
    { 0 },
    { 1.0 / 5 },
    { 3.0 / 40, 9.0 / 40 },
    { 44.0 / 45, -56.0 / 15, 32.0 / 9 },
    { 19372.0 / 6561, -25360.0 / 2187, 64448.0 / 6561, -212.0 / 729 },
    { 9017.0 / 3168, -355.0 / 33, 46732.0 / 5247, 49.0 / 176, -5103.0 / 18656 },
    { 35.0 / 384, 0, 500.0 / 1113, 125.0 / 192, -2187.0 / 6784, 11.0 / 84 } };
static const double DP_E[7] = { 71.0 / 57600, 0, -71.0 / 16695, 71.0 / 1920, -17253.0 / 339200, 22.0 / 525, -1.0 / 40 };

void mo_dopri5_tableau(double a[42], double e[7])
{
    for (int i = 0; i < 7; i++) for (int j = 0; j < 6; j++) a[i * 6 + j] = DP_A[i][j];
    for (int i = 0; i < 7; i++) e[i] = DP_E[i];
}

/* One step. RK4: classical + projection (tol ignored, err = 0). DOPRI5: DESIGN.md R8:
 * k1..k6, y5 = m + dt sum b5_j k_j, k7 = f(y5), E = dt sum e_j k_j, err = max_i |E_i|,
 * accept iff tol<=0 or err<=tol; on accept m <- y5/|y5|, t += dt;
 * dt_next = dt*clamp(0.9 (tol/err)^(1/5), 0.2, 5) (5 if err = 0); tol<=0: dt_next = dt. */
static int step_inner(mo_sim *s, double *m, double dt, double tol, int *accepted, double *err_out, double *dt_next, double *max_dmdt)
{
    const long N = s->N, n3 = 3 * N;
    int rc = 0;
    if (s->integrator == 2) {
        rc = cayley_step(s, m, dt, max_dmdt);
        if (accepted) *accepted = 1;
        if (err_out) *err_out = 0;
        if (dt_next) *dt_next = dt;
        return rc;
    }
    if (s->integrator == 0) {
        double *k = (double *)malloc(sizeof(double) * n3 * 4), *y = (double *)malloc(sizeof(double) * n3);
        s->t_eval = s->t;
        if ((rc = mo_llg_rhs(s, m, k))) goto done4;
        for (long q = 0; q < n3; q++) y[q] = m[q] + 0.5 * dt * k[q];
        s->t_eval = s->t + 0.5 * dt;
        if ((rc = mo_llg_rhs(s, y, k + n3))) goto done4;
        for (long q = 0; q < n3; q++) y[q] = m[q] + 0.5 * dt * k[n3 + q];
        if ((rc = mo_llg_rhs(s, y, k + 2 * n3))) goto done4;
        for (long q = 0; q < n3; q++) y[q] = m[q] + dt * k[2 * n3 + q];
        s->t_eval = s->t + dt;
        if ((rc = mo_llg_rhs(s, y, k + 3 * n3))) goto done4;
        if (max_dmdt) *max_dmdt = max_norm(s, k);
        for (long q = 0; q < n3; q++) m[q] += dt / 6.0 * (k[q] + 2 * k[n3 + q] + 2 * k[2 * n3 + q] + k[3 * n3 + q]);
        project(s, m);
        s->t += dt;
        if (accepted) *accepted = 1;
        if (err_out) *err_out = 0;
        if (dt_next) *dt_next = dt;
    done4:
        free(k); free(y);
        return rc;
    }
    double *k = (double *)malloc(sizeof(double) * n3 * 7), *y = (double *)malloc(sizeof(double) * n3);
    for (int st = 0; st < 7; st++) {
        for (long q = 0; q < n3; q++) {
            double acc = 0;
            for (int j = 0; j < st; j++) acc += DP_A[st][j] * k[j * n3 + q];
            y[q] = m[q] + dt * acc;
        }
        {
            static const double DP_C[7] = { 0.0, 1.0 / 5, 3.0 / 10, 4.0 / 5, 8.0 / 9, 1.0, 1.0 };      /* row sums of DP_A */
            s->t_eval = s->t + DP_C[st] * dt;
        }
        if ((rc = mo_llg_rhs(s, y, k + st * n3))) goto done5;
    }
    /* y now holds y5 (stage-7 input) */
    {
        double *E = (double *)malloc(sizeof(double) * n3);
        for (long q = 0; q < n3; q++) {
            double acc = 0;
            for (int j = 0; j < 7; j++) acc += DP_E[j] * k[j * n3 + q];
            E[q] = dt * acc;
        }
        double err = max_norm(s, E);
        free(E);
        int ok = (tol <= 0) || (err <= tol);
        if (max_dmdt) *max_dmdt = max_norm(s, k);
        if (ok) { memcpy(m, y, sizeof(double) * n3); project(s, m); s->t += dt; }
        double dn = dt;
        if (tol > 0) {
            double fac = err == 0 ? 5.0 : 0.9 * pow(tol / err, 0.2);
            if (fac < 0.2) fac = 0.2;
            if (fac > 5.0) fac = 5.0;
            if (err != err) fac = 0.2;
            dn = dt * fac;
        }
        if (accepted) *accepted = ok;
        if (err_out) *err_out = err;
        if (dt_next) *dt_next = dn;
    }
done5:
    free(k); free(y);
    return rc;
}

/* The thermal field (Eq. 42) is drawn once per step attempt with that attempt's dt and held over its stages
 * ("an effective field can be incorporated into existing integrators"). */
int mo_step(mo_sim *s, double *m, double dt, double tol, int *accepted, double *err_out, double *dt_next, double *max_dmdt)
{
    double *xi = NULL;
    if (s->temperature > 0.0) {
        xi = (double *)malloc(sizeof(double) * 3 * s->N);
        mo_thermal_field(s, dt, s->th_step, xi);
        s->Hth = xi;
    }
    s->in_step = 1;
    int rc = step_inner(s, m, dt, tol, accepted, err_out, dt_next, max_dmdt);
    s->in_step = 0;
    s->Hth = NULL;
    if (xi) { s->th_step++; free(xi); }
    return rc;
}

/* relax: adaptive steps until max|dm/dt| < stop_dmdt or max_steps */
int mo_relax(mo_sim *s, double *m, double tol, double stop_dmdt, long max_steps, double dt0, long *steps_done, double *max_dmdt_out)
{
    double dt = dt0, md = INFINITY;
    long it = 0;
    for (; it < max_steps; it++) {
        int ok; double err, dn;
        int rc = mo_step(s, m, dt, tol, &ok, &err, &dn, &md);
        if (rc) return rc;
        dt = dn;
        if (md < stop_dmdt) { it++; break; }
    }
    if (steps_done) *steps_done = it;
    if (max_dmdt_out) *max_dmdt_out = md;
    return 0;
}

/* ------------------------------------------------------------------------------------
 * Steepest-descent energy minimisation with Barzilai-Borwein steps, PAPER.md:376-393 (§VI).
 *   f_k = m_k x H_eff(m_k),  g_k = m_k x (m_k x H_eff(m_k))            (text under Eq. 51)
 *   (1 + tau^2 f_k^2 / 4) m_{k+1} = (1 - tau^2 f_k^2 / 4) m_k - tau g_k      (Eq. 51, per cell)
 *   s_{k-1} = m_k - m_{k-1},  y_{k-1} = g_k - g_{k-1}
 *   tau^1 = sum_i s.s / sum_i s.y ,  tau^2 = sum_i s.y / sum_i y.y           (Eq. 52, sums over cells)
 * Readings where the paper is silent (R16): the first step uses the caller's tau0; afterwards
 * tau^1 on odd k and tau^2 on even k (the alternation of ref [44]); |tau| is used, clamped to
 * [tau_min, tau_max]; a vanishing or non-finite quotient falls back to tau0; iteration stops BEFORE the
 * update when max_i |g_k,i| < stop_torque (A/m) or after max_steps updates.  Cells with Ms = 0 are
 * left untouched and do not enter the sums.  No projection: Eq. 50 preserves |m| by itself.
 * mo_sd_update is the single update of Eq. 51 with a given tau (exposed for the pins). */
void mo_sd_update(const mo_sim *s, double *m, const double *H, double tau)
{
    const long N = s->N;
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) continue;
        const double mx = m[q], my = m[N + q], mz = m[2 * N + q];
        const double hx = H[q], hy = H[N + q], hz = H[2 * N + q];
        const double fx = my * hz - mz * hy, fy = mz * hx - mx * hz, fz = mx * hy - my * hx;       /* f = m x H */
        const double gx = my * fz - mz * fy, gy = mz * fx - mx * fz, gz = mx * fy - my * fx;       /* g = m x f */
        const double a = 0.25 * tau * tau * (fx * fx + fy * fy + fz * fz);
        m[q] = ((1.0 - a) * mx - tau * gx) / (1.0 + a);
        m[N + q] = ((1.0 - a) * my - tau * gy) / (1.0 + a);
        m[2 * N + q] = ((1.0 - a) * mz - tau * gz) / (1.0 + a);
    }
}

int mo_minimize(mo_sim *s, double *m, double tau0, double tau_min, double tau_max, double stop_torque, long max_steps,
                long *steps_done, double *max_torque_out, double *tau_last)
{
    const long N = s->N;
    double *H = (double *)malloc(sizeof(double) * 3 * N), *g = (double *)malloc(sizeof(double) * 3 * N);
    double *gp = (double *)malloc(sizeof(double) * 3 * N), *mp = (double *)malloc(sizeof(double) * 3 * N);
    double tau = tau0, maxg = INFINITY;
    long k = 0;
    int rc = 0;
    for (;; k++) {
        if ((rc = mo_effective_field(s, m, H))) break;
        maxg = 0.0;
        for (long q = 0; q < N; q++) {
            double gx = 0, gy = 0, gz = 0;
            if (s->Ms[q] != 0.0) {
                const double mx = m[q], my = m[N + q], mz = m[2 * N + q];
                const double hx = H[q], hy = H[N + q], hz = H[2 * N + q];
                const double fx = my * hz - mz * hy, fy = mz * hx - mx * hz, fz = mx * hy - my * hx;
                gx = my * fz - mz * fy; gy = mz * fx - mx * fz; gz = mx * fy - my * fx;
                const double n = sqrt(gx * gx + gy * gy + gz * gz);
                if (!(n <= maxg)) maxg = n;      /* keeps a NaN */
            }
            g[q] = gx; g[N + q] = gy; g[2 * N + q] = gz;
        }
        if (!(maxg == maxg)) { rc = -6; break; }
        if (maxg < stop_torque || k >= max_steps) break;
        if (k > 0) {                              /* Eq. 52 */
            double ss = 0, sy = 0, yy = 0;
            for (long q = 0; q < N; q++) {
                if (s->Ms[q] == 0.0) continue;
                for (int c = 0; c < 3; c++) {
                    const double sv = m[c * N + q] - mp[c * N + q], yv = g[c * N + q] - gp[c * N + q];
                    ss += sv * sv; sy += sv * yv; yy += yv * yv;
                }
            }
            double t = (k & 1) ? ss / sy : sy / yy;
            t = fabs(t);
            if (!(t > 0.0) || isinf(t)) t = tau0;
            tau = t < tau_min ? tau_min : (t > tau_max ? tau_max : t);
        }
        memcpy(mp, m, sizeof(double) * 3 * N);
        memcpy(gp, g, sizeof(double) * 3 * N);
        mo_sd_update(s, m, H, tau);               /* Eq. 51 */
    }
    if (steps_done) *steps_done = k;
    if (max_torque_out) *max_torque_out = maxg;
    if (tau_last) *tau_last = tau;
    free(H); free(g); free(gp); free(mp);
    return rc;
}

/* E = - mu0 sum_i V Ms_i m_i . (1/2 H_d + 1/2 H_ex + 1/2 H_dmi + 1/2 H_an + H_ext)_i
 * terms: demag, exchange, dmi, anisotropy, zeeman.  (Quadratic terms carry 1/2, Eq. 1.) */
int mo_energy(mo_sim *s, const double *m, double *E_total, double E_terms[5])
{
    const long N = s->N;
    double *H = (double *)malloc(sizeof(double) * 3 * N);
    /* quadratic terms carry 1/2, the quartic cubic-anisotropy term 1/4 (Euler), the linear Zeeman term 1;
     * cubic anisotropy is reported inside the anisotropy slot */
    const int bits[6] = { 16, 1, 2, 4, 8, 32 };
    const double w[6] = { 0.5, 0.5, 0.5, 0.5, 1.0, 0.25 };
    const int slot[6] = { 0, 1, 2, 3, 4, 3 };
    const double V = s->dx * s->dy * s->dz;
    double tot = 0;
    if (E_terms) for (int t = 0; t < 5; t++) E_terms[t] = 0.0;
    for (int t = 0; t < 6; t++) {
        if (t == 5 && s->Kc == 0.0) continue;
        int rc = mo_field_terms(s, m, H, bits[t]);
        if (rc) { free(H); return rc; }
        double e = 0;
        for (long q = 0; q < N; q++)
            e += s->Ms[q] * (m[q] * H[q] + m[N + q] * H[N + q] + m[2 * N + q] * H[2 * N + q]);
        e *= -MO_MU0 * V * w[t];
        if (E_terms) E_terms[slot[t]] += e;
        tot += e;
    }
    if (E_total) *E_total = tot;
    free(H);
    return 0;
}

int mo_average_m(mo_sim *s, const double *m, double out3[3])
{
    const long N = s->N;
    long cnt = 0;
    double a[3] = { 0, 0, 0 };
    for (long q = 0; q < N; q++) {
        if (s->Ms[q] == 0.0) continue;
        cnt++;
        for (int c = 0; c < 3; c++) a[c] += m[c * N + q];
    }
    for (int c = 0; c < 3; c++) out3[c] = cnt ? a[c] / (double)cnt : 0.0;
    return 0;
}

/* ---------------------------------------------------------------------------------- */
int mo_create(mo_sim **out, int nx, int ny, int nz, double dx, double dy, double dz)
{
    if (!out || nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0)) return -1;
    mo_sim *s = (mo_sim *)calloc(1, sizeof(mo_sim));
    s->nx = nx; s->ny = ny; s->nz = nz; s->dx = dx; s->dy = dy; s->dz = dz;
    s->N = (long)nx * ny * nz;
    s->Ms = (double *)calloc(s->N, sizeof(double));
    s->gamma = 2.211e5; s->alpha = 0.5; s->uz = 1.0; s->integrator = 1; s->demag = 1;
    s->px = nx > 1 ? 2 * nx : 1; s->py = ny > 1 ? 2 * ny : 1; s->pz = nz > 1 ? 2 * nz : 1;
    *out = s;
    return 0;
}

int mo_destroy(mo_sim *s)
{
    if (!s) return 0;
    free(s->Ms); free(s->Nten); free(s->Khat); free(s->Acell); free(s->Dcell); free(s->Hcell); free(s);
    return 0;
}

int mo_set_Ms_uniform(mo_sim *s, double Ms) { for (long q = 0; q < s->N; q++) s->Ms[q] = Ms; return 0; }
int mo_set_Ms(mo_sim *s, const double *Ms) { memcpy(s->Ms, Ms, sizeof(double) * s->N); return 0; }
int mo_set_A(mo_sim *s, double A) { s->A = A; return 0; }
int mo_set_D(mo_sim *s, double D, int kind) { if (kind < 0 || kind > 3) return -1; s->D = D; s->dmi_kind = kind; return 0; }
int mo_set_Ku(mo_sim *s, double Ku) { s->Ku = Ku; return 0; }
int mo_set_Kc(mo_sim *s, double Kc) { s->Kc = Kc; return 0; }
static int set_cell_array(double **dst, const double *src, long n)
{
    free(*dst); *dst = NULL;
    if (src) { *dst = (double *)malloc(sizeof(double) * n); memcpy(*dst, src, sizeof(double) * n); }
    return 0;
}
/* cell-based constants (NULL: back to the uniform value) */
int mo_set_A_cell(mo_sim *s, const double *A) { return set_cell_array(&s->Acell, A, s->N); }
int mo_set_D_cell(mo_sim *s, const double *D, int kind) { if (kind < 0 || kind > 3) return -1; s->dmi_kind = kind; return set_cell_array(&s->Dcell, D, s->N); }
int mo_set_H_ext_cell(mo_sim *s, const double *H) { return set_cell_array(&s->Hcell, H, 3 * s->N); }
int mo_set_axis(mo_sim *s, double ux, double uy, double uz)
{
    if (ux == 0 && uy == 0 && uz == 0) return -1;
    s->ux = ux; s->uy = uy; s->uz = uz; return 0;
}
int mo_set_H_ext(mo_sim *s, double hx, double hy, double hz) { s->hx = hx; s->hy = hy; s->hz = hz; return 0; }
int mo_set_alpha(mo_sim *s, double a) { s->alpha = a; return 0; }
int mo_set_gamma(mo_sim *s, double g) { s->gamma = g; return 0; }
int mo_set_integrator(mo_sim *s, int i) { if (i < 0 || i > 2) return -1; s->integrator = i; return 0; }
int mo_set_zhang_li(mo_sim *s, double ux, double uy, double uz, double beta)
{
    s->stt_u[0] = ux; s->stt_u[1] = uy; s->stt_u[2] = uz; s->stt_beta = beta;
    s->stt_on = (ux != 0.0 || uy != 0.0 || uz != 0.0);
    return 0;
}
int mo_set_zhang_li_pulse(mo_sim *s, double b, double w) { s->stt_b = b; s->stt_w = w; return 0; }
int mo_set_slonczewski(mo_sim *s, double aJ, double bJ, double px, double py, double pz)
{
    const double n = sqrt(px * px + py * py + pz * pz);
    s->sl_on = (aJ != 0.0 || bJ != 0.0);
    if (s->sl_on && !(n > 0)) return -1;
    s->sl_aJ = aJ; s->sl_bJ = bJ;
    s->sl_p[0] = n > 0 ? px / n : 0; s->sl_p[1] = n > 0 ? py / n : 0; s->sl_p[2] = n > 0 ? pz / n : 0;
    return 0;
}
int mo_set_temperature(mo_sim *s, double T, unsigned long long seed)
{
    if (!(T >= 0.0)) return -1;
    s->temperature = T; s->th_seed = seed; s->th_step = 0;
    return 0;
}
/* 0 off, 1 FFT path, 2 direct O(N^2) */
int mo_set_demag(mo_sim *s, int mode) { if (mode < 0 || mode > 2) return -1; s->demag = mode; return 0; }
double mo_time(const mo_sim *s) { return s->t; }
int mo_set_time(mo_sim *s, double t) { s->t = t; return 0; }

int mo_init_demag(mo_sim *s)
{
    if (!s->Nten) {
        s->Nten = (double *)malloc(sizeof(double) * 6 * s->N);
        mo_newell_tensor(s->nx, s->ny, s->nz, s->dx, s->dy, s->dz, s->Nten);
    }
    return 0;
}

/* real-space tensor component (0..5 = xx,yy,zz,xy,xz,yz) at offsets i,j,k >= 0; N doubles */
int mo_get_demag_kernel(mo_sim *s, int comp, double *out)
{
    if (!s->Nten) return -3;
    if (comp < 0 || comp > 5) return -1;
    memcpy(out, s->Nten + (size_t)comp * s->N, sizeof(double) * s->N);
    return 0;
}

/* imaginary-part check of the cached spectrum: max |Im Khat| / max |Khat| (pin: vanishes) */
double mo_khat_imag_ratio(mo_sim *s)
{
    if (!s->Nten) return -1;
    if (!s->Khat) build_khat(s);
    const long P = (long)s->px * s->py * s->pz;
    double mi = 0, ma = 0;
    for (long q = 0; q < 6 * P; q++) {
        double re = fabs(s->Khat[2 * q]), im = fabs(s->Khat[2 * q + 1]);
        if (im > mi) mi = im;
        if (re > ma) ma = re;
    }
    return mi / ma;
}
