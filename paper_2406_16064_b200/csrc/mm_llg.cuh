// mm_llg.cuh — per-cell arithmetic of the fused local-field / LL-torque / RK-stage kernel.
//   exchange  Eq. 5      DMI  Eq. 15
//   anisotropy Eq. 32 continuum reading (R6)   Zeeman Eq. 35
//   LL torque Eq. 37;  RK stage algebra: DESIGN.md R8
// A neighbour is absent when outside the mesh or when its Ms is 0 (R4); Ms_i = 0 => H = 0, k = 0 (R5).
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"

namespace mm {

template <typename T> struct LocalP {
    T cex[3];      // 2A/(mu0 d_a^2)
    T cdm[3];      // D/(mu0 d_a)
    T cku;         // 2Ku/mu0
    T u[3];        // unit axis
    T hext[3];
    T gp, agp;     // gamma/(1+alpha^2), alpha*gamma/(1+alpha^2)
    int dmi;       // 0 none, 1 bulk, 2 interfacial
    int terms;     // bit0 exchange, bit1 DMI, bit2 anisotropy, bit3 Zeeman, bit4 demag
};

template <typename T> struct v3 { T x, y, z; };
template <typename T> MM_HD v3<T> ld3(const T* p, long N, long q) { v3<T> r; r.x = p[q]; r.y = p[N + q]; r.z = p[2 * N + q]; return r; }

// H_eff at cell (i,j,k) given H_d (or 0).  y = stage magnetisation.
template <typename T>
MM_HD v3<T> local_field(const Geom& g, const LocalP<T>& lp, const T* __restrict__ y, const T* __restrict__ Ms,
                        int i, int j, int k, long q, T Msi, v3<T> mi, v3<T> H)
{
    const long N = g.N;
    const T inv = (T)1 / Msi;
    if ((lp.terms & 3) != 0) {
        v3<T> ex = { 0, 0, 0 };           // sum_a cex_a sum_{+-} (m_j - m_i)
        v3<T> S[3];                        // S_a = m_{+a} - m_{-a} over present neighbours
        const long str[3] = { 1, g.nx, (long)g.nx * g.ny };
        const int pos[3] = { i, j, k }, lim[3] = { g.nx, g.ny, g.nz };
#pragma unroll
        for (int a = 0; a < 3; a++) {
            v3<T> sm = { 0, 0, 0 };
            v3<T> acc = { 0, 0, 0 };
            if (pos[a] > 0) {
                const long p = q - str[a];
                if (Ms[p] != (T)0) {
                    const v3<T> mj = ld3(y, N, p);
                    acc.x += mj.x - mi.x; acc.y += mj.y - mi.y; acc.z += mj.z - mi.z;
                    sm.x -= mj.x; sm.y -= mj.y; sm.z -= mj.z;
                }
            }
            if (pos[a] < lim[a] - 1) {
                const long p = q + str[a];
                if (Ms[p] != (T)0) {
                    const v3<T> mj = ld3(y, N, p);
                    acc.x += mj.x - mi.x; acc.y += mj.y - mi.y; acc.z += mj.z - mi.z;
                    sm.x += mj.x; sm.y += mj.y; sm.z += mj.z;
                }
            }
            ex.x += lp.cex[a] * acc.x; ex.y += lp.cex[a] * acc.y; ex.z += lp.cex[a] * acc.z;
            S[a] = sm;
        }
        if (lp.terms & 1) { H.x += inv * ex.x; H.y += inv * ex.y; H.z += inv * ex.z; }
        if ((lp.terms & 2) && lp.dmi != 0) {
            v3<T> d;
            if (lp.dmi == 1) {      // bulk: e_ij = r^_ij  =>  sum_a cdm_a (a^ x S_a)
                d.x = lp.cdm[1] * S[1].z - lp.cdm[2] * S[2].y;
                d.y = -lp.cdm[0] * S[0].z + lp.cdm[2] * S[2].x;
                d.z = lp.cdm[0] * S[0].y - lp.cdm[1] * S[1].x;
            } else {                // interfacial: e_ij = z^ x r^_ij : (y^ x S_x) - (x^ x S_y)
                d.x = lp.cdm[0] * S[0].z;
                d.y = lp.cdm[1] * S[1].z;
                d.z = -lp.cdm[0] * S[0].x - lp.cdm[1] * S[1].y;
            }
            H.x -= inv * d.x; H.y -= inv * d.y; H.z -= inv * d.z;
        }
    }
    if (lp.terms & 4) {
        const T f = inv * lp.cku * (mi.x * lp.u[0] + mi.y * lp.u[1] + mi.z * lp.u[2]);
        H.x += f * lp.u[0]; H.y += f * lp.u[1]; H.z += f * lp.u[2];
    }
    if (lp.terms & 8) { H.x += lp.hext[0]; H.y += lp.hext[1]; H.z += lp.hext[2]; }
    return H;
}

template <typename T> MM_HD v3<T> ll_torque(const LocalP<T>& lp, v3<T> m, v3<T> H)
{
    const T ax = m.y * H.z - m.z * H.y, ay = m.z * H.x - m.x * H.z, az = m.x * H.y - m.y * H.x;
    const T bx = m.y * az - m.z * ay, by = m.z * ax - m.x * az, bz = m.x * ay - m.y * ax;
    v3<T> k;
    k.x = -lp.gp * ax - lp.agp * bx;
    k.y = -lp.gp * ay - lp.agp * by;
    k.z = -lp.gp * az - lp.agp * bz;
    return k;
}

}  // namespace mm
