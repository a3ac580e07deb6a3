// mm_llg.cuh — per-cell arithmetic of the fused local-field / LL-torque / RK-stage kernel.
//   exchange  Eq. 5      DMI  Eq. 15
//   anisotropy Eq. 32 continuum reading (R6)   Zeeman Eq. 35
//   cell-based A and D: A_ij = 2 A_i A_j / (A_i + A_j), D_ij likewise; D2d DMI table
//   (Eq. 14); cubic anisotropy Eq. 33-34 continuum reading (R6);
//   per-cell external field (Eq. 35 with H_i)
//   LL torque Eq. 37;  RK stage algebra: DESIGN.md R8
// A neighbour is absent when outside the mesh or when its Ms is 0 (R4); Ms_i = 0 => H = 0, k = 0 (R5).
#pragma once
#include "mm_fft.cuh"
#include "mm_kernels.cuh"

namespace mm {

template <typename T> struct LocalP {
    T cex[3];      // 2A/(mu0 d_a^2)   (2/(mu0 d_a^2) when A is cell-based: the bond value A_ij multiplies it)
    T cdm[3];      // D/(mu0 d_a)      (1/(mu0 d_a) when D is cell-based)
    T cku;         // 2Ku/mu0
    T ckc;         // 4Kc/mu0 (cubic anisotropy, crystal axes = mesh axes)
    T u[3];        // unit axis
    T hext[3];
    T gp, agp;     // gamma/(1+alpha^2), alpha*gamma/(1+alpha^2)
    int dmi;       // 0 none, 1 bulk, 2 interfacial, 3 D2d
    int terms;     // bit0 exchange, bit1 DMI, bit2 uniaxial anisotropy, bit3 Zeeman, bit4 demag, bit5 cubic anisotropy
    const T* Acell;   // N per-cell exchange constants or nullptr (uniform A)
    const T* Dcell;   // N per-cell DMI constants or nullptr (uniform D)
    const T* Hcell;   // 3N per-cell external field (SoA) or nullptr (uniform hext)
    // torque extensions and thermal field (general kernels only)
    const T* Hth;     // 3N thermal field of the step in progress (Eq. 42) or nullptr
    T stt[3];         // Zhang-Li: u_a / (2 Delta_a)  (central differences of (u.grad) m)
    T beta;           // Zhang-Li non-adiabaticity
    T sl_a, sl_b;     // Slonczewski / SOT written as a field: a_J / gamma, b_J / gamma
    T p[3];           // unit polarisation vector
    T gam, al;        // gamma, alpha (f of Eq. 44 and f_stt need them separately)
    int stt_on, sl_on;
    double stt_b, stt_w;   // time profile of the Zhang-Li current: u(t) = u exp(-b t) cos(w t); 0, 0 = constant
};

// bond value of a cell-based constant: harmonic mean, 0 when both vanish
template <typename T> MM_HD T harm(T a, T b) { const T s = a + b; return s != (T)0 ? (T)2 * a * b / s : (T)0; }

template <typename T> struct v3 { T x, y, z; };
template <typename T> MM_HD v3<T> ld3(const T* p, long N, long q) { v3<T> r; r.x = p[q]; r.y = p[N + q]; r.z = p[2 * N + q]; return r; }

// anisotropy + Zeeman part of H_eff (inv = 1/Ms_i); hext = the external field of this cell
template <typename T> MM_HD v3<T> local_field_rest(const LocalP<T>& lp, T inv, v3<T> mi, v3<T> H, v3<T> hext)
{
    if (lp.terms & 4) {
        const T f = inv * lp.cku * (mi.x * lp.u[0] + mi.y * lp.u[1] + mi.z * lp.u[2]);
        H.x += f * lp.u[0]; H.y += f * lp.u[1]; H.z += f * lp.u[2];
    }
    if (lp.terms & 32) {     // Eq. 33: w = Kc (mx^4 + my^4 + mz^4)  =>  H = -(4Kc/(mu0 Ms)) (mx^3, my^3, mz^3)
        const T f = -inv * lp.ckc;
        H.x += f * mi.x * mi.x * mi.x; H.y += f * mi.y * mi.y * mi.y; H.z += f * mi.z * mi.z * mi.z;
    }
    if (lp.terms & 8) { H.x += hext.x; H.y += hext.y; H.z += hext.z; }
    return H;
}
template <typename T> MM_HD v3<T> local_field_rest(const LocalP<T>& lp, T inv, v3<T> mi, v3<T> H)
{
    const v3<T> h = { lp.hext[0], lp.hext[1], lp.hext[2] };
    return local_field_rest<T>(lp, inv, mi, H, h);
}

// H_eff from the six neighbour values nb[-x,+x,-y,+y,-z,+z] (ok[] = neighbour present) added to H
// GEN: cell-based A and / or D — wA[b], wD[b] are the bond values A_ij, D_ij towards neighbour b (1 for a constant
// that is uniform: it is then inside cex / cdm).
template <typename T> MM_HD v3<T> cross(v3<T> a, v3<T> b)
{
    v3<T> c = { a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x };
    return c;
}

// tau = (u.grad) m by central differences; an absent neighbour is replaced by the cell itself (R17)
template <typename T> MM_HD v3<T> stt_tau(const LocalP<T>& lp, v3<T> mi, const v3<T>* nb, const bool* ok)
{
    v3<T> t = { 0, 0, 0 };
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const v3<T> lo = ok[2 * a] ? nb[2 * a] : mi, hi = ok[2 * a + 1] ? nb[2 * a + 1] : mi;
        t.x += lp.stt[a] * (hi.x - lo.x); t.y += lp.stt[a] * (hi.y - lo.y); t.z += lp.stt[a] * (hi.z - lo.z);
    }
    return t;
}

// f_stt = [(beta - alpha) tau + (1 + alpha beta) m x tau] / (1 + alpha^2)
template <typename T> MM_HD v3<T> stt_f(const LocalP<T>& lp, v3<T> m, v3<T> tau)
{
    const v3<T> mt = cross<T>(m, tau);
    const T den = (T)1 / ((T)1 + lp.al * lp.al), c1 = (lp.beta - lp.al) * den, c2 = ((T)1 + lp.al * lp.beta) * den;
    v3<T> f = { c1 * tau.x + c2 * mt.x, c1 * tau.y + c2 * mt.y, c1 * tau.z + c2 * mt.z };
    return f;
}

// Eq. 40 folded into the field: H + (a_J / gamma) m x p + (b_J / gamma) p
template <typename T> MM_HD v3<T> add_slonczewski(const LocalP<T>& lp, v3<T> m, v3<T> H)
{
    const v3<T> p = { lp.p[0], lp.p[1], lp.p[2] };
    const v3<T> mp = cross<T>(m, p);
    H.x += lp.sl_a * mp.x + lp.sl_b * p.x; H.y += lp.sl_a * mp.y + lp.sl_b * p.y; H.z += lp.sl_a * mp.z + lp.sl_b * p.z;
    return H;
}

// f of Eq. 44: gamma (H + alpha m x H) / (1 + alpha^2)
template <typename T> MM_HD v3<T> llg_f(const LocalP<T>& lp, v3<T> m, v3<T> H)
{
    const v3<T> mH = cross<T>(m, H);
    v3<T> f = { lp.gp * (H.x + lp.al * mH.x), lp.gp * (H.y + lp.al * mH.y), lp.gp * (H.z + lp.al * mH.z) };
    return f;
}

// Eq. 49: d omega / dt = f - (omega x f) / 2 + (omega . f) omega / 4
template <typename T> MM_HD v3<T> cayley_domega(v3<T> w, v3<T> f)
{
    const v3<T> wf = cross<T>(w, f);
    const T d = (T)0.25 * (w.x * f.x + w.y * f.y + w.z * f.z);
    v3<T> r = { f.x - (T)0.5 * wf.x + d * w.x, f.y - (T)0.5 * wf.y + d * w.y, f.z - (T)0.5 * wf.z + d * w.z };
    return r;
}

// Eq. 43, 47 in closed vector form: Q(omega) m = m + (omega x m + omega x (omega x m) / 2) / (1 + |omega|^2 / 4)
template <typename T> MM_HD v3<T> cayley_apply(v3<T> w, v3<T> m)
{
    const v3<T> wm = cross<T>(w, m), wwm = cross<T>(w, wm);
    const T s = (T)1 / ((T)1 + (T)0.25 * (w.x * w.x + w.y * w.y + w.z * w.z));
    v3<T> r = { m.x + s * (wm.x + (T)0.5 * wwm.x), m.y + s * (wm.y + (T)0.5 * wwm.y), m.z + s * (wm.z + (T)0.5 * wwm.z) };
    return r;
}

template <typename T, bool GEN = false>
MM_HD v3<T> local_field_nb(const LocalP<T>& lp, T inv, v3<T> mi, const v3<T>* nb, const bool* ok, v3<T> H, v3<T> hext,
                           const T* wA = nullptr, const T* wD = nullptr)
{
    v3<T> ex = { 0, 0, 0 };           // sum_a cex_a sum_{+-} (m_j - m_i)
    v3<T> S[3];                        // S_a = m_{+a} - m_{-a} over present neighbours
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const v3<T> mm_ = nb[2 * a], mp = nb[2 * a + 1];
        const bool bm = ok[2 * a], bp = ok[2 * a + 1];
        T dmx = bm ? mm_.x - mi.x : (T)0, dmy = bm ? mm_.y - mi.y : (T)0, dmz = bm ? mm_.z - mi.z : (T)0;
        T dpx = bp ? mp.x - mi.x : (T)0, dpy = bp ? mp.y - mi.y : (T)0, dpz = bp ? mp.z - mi.z : (T)0;
        if (GEN) {
            const T am = wA[2 * a], ap = wA[2 * a + 1];
            dmx *= am; dmy *= am; dmz *= am; dpx *= ap; dpy *= ap; dpz *= ap;
        }
        ex.x += lp.cex[a] * (dmx + dpx); ex.y += lp.cex[a] * (dmy + dpy); ex.z += lp.cex[a] * (dmz + dpz);
        if (GEN) {
            const T bm_ = bm ? wD[2 * a] : (T)0, bp_ = bp ? wD[2 * a + 1] : (T)0;
            S[a].x = bp_ * mp.x - bm_ * mm_.x; S[a].y = bp_ * mp.y - bm_ * mm_.y; S[a].z = bp_ * mp.z - bm_ * mm_.z;
        } else {
            S[a].x = (bp ? mp.x : (T)0) - (bm ? mm_.x : (T)0);
            S[a].y = (bp ? mp.y : (T)0) - (bm ? mm_.y : (T)0);
            S[a].z = (bp ? mp.z : (T)0) - (bm ? mm_.z : (T)0);
        }
    }
    if (lp.terms & 1) { H.x += inv * ex.x; H.y += inv * ex.y; H.z += inv * ex.z; }
    if ((lp.terms & 2) && lp.dmi != 0) {
        v3<T> d;
        if (lp.dmi == 1) {      // bulk: e_ij = r^_ij  =>  sum_a cdm_a (a^ x S_a)
            d.x = lp.cdm[1] * S[1].z - lp.cdm[2] * S[2].y;
            d.y = -lp.cdm[0] * S[0].z + lp.cdm[2] * S[2].x;
            d.z = lp.cdm[0] * S[0].y - lp.cdm[1] * S[1].x;
        } else if (lp.dmi == 2) {   // interfacial: e_ij = z^ x r^_ij : (y^ x S_x) - (x^ x S_y)
            d.x = lp.cdm[0] * S[0].z;
            d.y = lp.cdm[1] * S[1].z;
            d.z = -lp.cdm[0] * S[0].x - lp.cdm[1] * S[1].y;
        } else {                // D2d: e_ij = {+x^, -x^, -y^, +y^, 0, 0} : -(x^ x S_x) + (y^ x S_y)
            d.x = lp.cdm[1] * S[1].z;
            d.y = lp.cdm[0] * S[0].z;
            d.z = -lp.cdm[0] * S[0].y - lp.cdm[1] * S[1].x;
        }
        H.x -= inv * d.x; H.y -= inv * d.y; H.z -= inv * d.z;
    }
    return local_field_rest<T>(lp, inv, mi, H, hext);
}

// H_eff at cell (i,j,k) given H_d (or 0).  y = stage magnetisation.  Branch-free in the data: every
// neighbour is loaded (index clamped to the cell itself when outside the mesh) and then selected,
// so all loads of a thread are in flight together.
template <typename T>
MM_HD v3<T> local_field(const Geom& g, const LocalP<T>& lp, const T* __restrict__ y, const T* __restrict__ Ms,
                        int i, int j, int k, long q, T Msi, v3<T> mi, v3<T> H, v3<T>* tau = nullptr)
{
    const long N = g.N;
    const T inv = (T)1 / Msi;
    v3<T> hext = { lp.hext[0], lp.hext[1], lp.hext[2] };
    if (lp.Hcell != nullptr && (lp.terms & 8)) hext = ld3(lp.Hcell, N, q);
    if (lp.Hth != nullptr) {      // thermal field of the step in progress: added whatever the term mask says
        const v3<T> ht = ld3(lp.Hth, N, q);
        H.x += ht.x; H.y += ht.y; H.z += ht.z;
    }
    if (tau != nullptr) { tau->x = 0; tau->y = 0; tau->z = 0; }
    if ((lp.terms & 3) == 0 && !(lp.stt_on && tau != nullptr)) return local_field_rest<T>(lp, inv, mi, H, hext);
    const long str[3] = { 1, g.nx, (long)g.nx * g.ny };
    const int pos[3] = { i, j, k }, lim[3] = { g.nx, g.ny, g.nz };
    v3<T> nb[6];
    bool ok[6];
    const bool gen = lp.Acell != nullptr || lp.Dcell != nullptr;
    T wA[6], wD[6];
#pragma unroll
    for (int a = 0; a < 3; a++) {
        const bool im = pos[a] > 0, ip = pos[a] < lim[a] - 1;
        const long pm = im ? q - str[a] : q, pp = ip ? q + str[a] : q;
        ok[2 * a] = im && (Ms[pm] != (T)0);
        ok[2 * a + 1] = ip && (Ms[pp] != (T)0);
        nb[2 * a] = ld3(y, N, pm);
        nb[2 * a + 1] = ld3(y, N, pp);
        if (gen) {
            wA[2 * a] = lp.Acell ? harm<T>(lp.Acell[q], lp.Acell[pm]) : (T)1;
            wA[2 * a + 1] = lp.Acell ? harm<T>(lp.Acell[q], lp.Acell[pp]) : (T)1;
            wD[2 * a] = lp.Dcell ? harm<T>(lp.Dcell[q], lp.Dcell[pm]) : (T)1;
            wD[2 * a + 1] = lp.Dcell ? harm<T>(lp.Dcell[q], lp.Dcell[pp]) : (T)1;
        }
    }
    if (lp.stt_on && tau != nullptr) *tau = stt_tau<T>(lp, mi, nb, ok);
    if (gen) return local_field_nb<T, true>(lp, inv, mi, nb, ok, H, hext, wA, wD);
    return local_field_nb<T, false>(lp, inv, mi, nb, ok, H, hext);
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
