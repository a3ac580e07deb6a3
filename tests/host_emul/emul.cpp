// Host emulation of the demag convolution passes: compiles the __host__ __device__ kernel bodies of
// paper_2406_16064_b200/csrc with g++ and runs every CTA sequentially with one "thread"
// (tid = 0, nthr = 1).  TEST HARNESS ONLY — checks the index arithmetic of the kernels on a box
// without a GPU; it is not a product path and nothing in the package loads it.
#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>
#include "../../paper_2406_16064_b200/csrc/mm_kernels.cuh"
#include "../../paper_2406_16064_b200/csrc/mm_kernels2.cuh"
#include "../../paper_2406_16064_b200/csrc/mm_passAC.cuh"
#include "../../paper_2406_16064_b200/csrc/mm_passB7.cuh"
#include "../../paper_2406_16064_b200/csrc/mm_passB3.cuh"
#include "../../paper_2406_16064_b200/csrc/mm_passB4.cuh"
#include "../../paper_2406_16064_b200/csrc/mm_llg.cuh"

using namespace mm;

template <typename T> static std::vector<cx<T>> make_tw(int twN)
{
    std::vector<cx<T>> h(twN / 2 + 1);
    for (int k = 0; k <= twN / 2; k++) {
        long double a = -2.0L * 3.14159265358979323846264338327950288L * k / twN;
        h[k].x = (T)cosl(a); h[k].y = (T)sinl(a);
    }
    return h;
}

static Geom make_geom(int nx, int ny, int nz, int G, int CH, int TC)
{
    Geom g;
    memset(&g, 0, sizeof(g));
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.px = 2 * nx; g.py = 2 * ny; g.pz = nz > 1 ? 2 * nz : 1;
    g.lognx = ilog2(nx); g.logny = ilog2(ny); g.logpy = ilog2(g.py); g.logpz = ilog2(g.pz);
    g.N = (long)nx * ny * nz;
    g.G = G; g.CH = CH; g.TC = TC;
    g.xpad = G * nz <= 4 ? 1 : 0;      // the library's rule (configure() in mm_lib.cu)
    g.Lx = ((nx + 1 + TC - 1) / TC) * TC;
    g.plane = (long)ny * g.Lx; g.comp = (long)g.pz * g.plane;
    g.kplane = (long)(ny + 1) * g.Lx; g.kcomp = (long)(nz > 1 ? nz + 1 : 1) * g.kplane;
    return g;
}

// Kfull: real part of the 3-D DFT of the wrapped tensor, natural order, [6][pz][py][px] doubles.
template <typename T>
static void run(int ver, int nx, int ny, int nz, int G, int CH, int TC, const double* Kfull, const double* Ms, const double* m, double* Hd)
{
    Geom g = make_geom(nx, ny, nz, G, CH, TC);
    int twN = g.px > g.py ? g.px : g.py;
    if (g.pz > twN) twN = g.pz;
    auto twv = make_tw<T>(twN);
    twiddles<T> tw; tw.tw = twv.data(); tw.twN = twN;
    std::vector<T> Kh((size_t)6 * g.kcomp, 0);
    const int nkz = nz > 1 ? nz + 1 : 1;
    for (int c = 0; c < 6; c++)
        for (int kz = 0; kz < nkz; kz++)
            for (int ky = 0; ky <= ny; ky++)
                for (int xp = 0; xp <= nx; xp++) {
                    int kx = xp < nx ? (int)brev(xp, g.lognx) : nx;
                    Kh[(size_t)c * g.kcomp + (size_t)kz * g.kplane + (size_t)ky * g.Lx + xp] =
                        (T)Kfull[(((size_t)c * g.pz + kz) * g.py + ky) * g.px + kx];
                }
    std::vector<T> Kc(ny >= 16 ? (size_t)kc_elems(g) : 0);
    for (long i = 0; i < (long)Kc.size(); i++) kc_fill<T>(g, Kh.data(), Kc.data(), i);
    std::vector<T> mt(3 * g.N), Mst(g.N), Hdt(3 * g.N);
    for (long i = 0; i < 3 * g.N; i++) mt[i] = (T)m[i];
    for (long i = 0; i < g.N; i++) Mst[i] = (T)Ms[i];
    std::vector<cx<T>> S((size_t)3 * g.comp);
    memset(S.data(), 0, S.size() * sizeof(cx<T>));
    std::vector<cx<T>> smem((size_t)std::max(std::max(smemA_elems(g), smemA2_elems(g)), smemB_elems(g)) + 16);
    const int gridA = 3 * (ny / G), gridB = (g.Lx / TC) * g.pz;
    const double P = (double)g.px * g.py * g.pz;
    const bool a2 = ver >= 2 && nx >= 32 && nz <= 32, b2 = ver >= 2 && ny >= 16, b5 = (ver == 5 || ver == 7) && ny >= 16;      // ver 42 / 44 without room for the cluster form fall to y_conv_body2
    for (int b = 0; b < gridA; b++) {
        if (!a2) fwd_xz_body<T>(g, mt.data(), Mst.data(), S.data(), tw, smem.data(), b, 0, 1);
        else switch (nz) {
#define CASE_A(NZ) case NZ: if (NZ <= 4 && g.xpad) fwd_xz_body3<T, NZ, (NZ <= 4)>(g, mt.data(), Mst.data(), S.data(), tw, smem.data(), b, 0, 1); else fwd_xz_body3<T, NZ, false>(g, mt.data(), Mst.data(), S.data(), tw, smem.data(), b, 0, 1); break;
            CASE_A(1) CASE_A(2) CASE_A(4) CASE_A(8) CASE_A(16) CASE_A(32)
        }
    }
    const bool b7 = ver == 7 && TC == (sizeof(T) == 8 ? 2 : 4) && ny >= 16 && ny <= 1024;
    const bool b7n = ver == 7 && sizeof(T) == 4 && TC == 2 && ny >= 16 && ny <= 1024;      // fp32 with 2-column tiles (the library's ny = 512 form)
    unsigned long long* nobar = nullptr;
    constexpr int LOGTC7 = sizeof(T) == 8 ? 1 : 2;
    const bool b3 = ver == 3 && ny >= 16;
    std::vector<cx<T>> S2(b3 ? S.size() : 0);      // half-tile pass B writes a second spectrum buffer
    const int Q4 = ver == 42 ? 2 : (ver == 44 ? 4 : 0);      // cluster pass B: the Q CTAs of a cluster run one after the other
    const bool b4 = Q4 != 0 && g.py / Q4 >= 16;
    if (b4) {
        std::vector<std::vector<cx<T>>> tiles(Q4, std::vector<cx<T>>((size_t)smemB4_elems(g, Q4) + 16));
        cx<T>* tp[4] = { nullptr, nullptr, nullptr, nullptr };
        for (int qq = 0; qq < Q4; qq++) tp[qq] = tiles[qq].data();
        for (int b = 0; b < gridB; b++) {
            for (int qq = 0; qq < Q4; qq++) {
                if (Q4 == 2) { if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body4_compute<T, (sizeof(T) == 4 ? 2 : 1), 2>(g, S.data(), Kh.data(), tw, tp[qq], b, qq, 0, 1); else y_conv_body4_compute<T, 1, 2>(g, S.data(), Kh.data(), tw, tp[qq], b, qq, 0, 1); }
                else { if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body4_compute<T, (sizeof(T) == 4 ? 2 : 1), 4>(g, S.data(), Kh.data(), tw, tp[qq], b, qq, 0, 1); else y_conv_body4_compute<T, 1, 4>(g, S.data(), Kh.data(), tw, tp[qq], b, qq, 0, 1); }
            }
            for (int qq = 0; qq < Q4; qq++) {
                if (Q4 == 2) { if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body4_combine<T, (sizeof(T) == 4 ? 2 : 1), 2>(g, S.data(), tp, b, qq, 0, 1); else y_conv_body4_combine<T, 1, 2>(g, S.data(), tp, b, qq, 0, 1); }
                else { if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body4_combine<T, (sizeof(T) == 4 ? 2 : 1), 4>(g, S.data(), tp, b, qq, 0, 1); else y_conv_body4_combine<T, 1, 4>(g, S.data(), tp, b, qq, 0, 1); }
            }
        }
    }
    for (int b = 0; b < gridB && !b4; b++) {
        if (b3) {
            if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body3<T, (sizeof(T) == 4 ? 2 : 1)>(g, S.data(), S2.data(), Kh.data(), tw, smem.data(), b, 0, 1);
            else y_conv_body3<T, 1>(g, S.data(), S2.data(), Kh.data(), tw, smem.data(), b, 0, 1);
        } else if (b7n) {
            switch (g.logny * 2 + (nz > 1)) {
#define CASE_B7N(L) case 2 * L: y_conv_body7<L, 1, false, 1, T>(g, S.data(), Kc.data(), tw, ilog2(twN), smem.data(), b, 0, 1, nullptr, nobar, nullptr); break; \
                    case 2 * L + 1: y_conv_body7<L, 1, true, 1, T>(g, S.data(), Kc.data(), tw, ilog2(twN), smem.data(), b, 0, 1, nullptr, nobar, nullptr); break;
                CASE_B7N(4) CASE_B7N(5) CASE_B7N(6) CASE_B7N(7) CASE_B7N(8) CASE_B7N(9) CASE_B7N(10)
            }
        } else if (b7) {
            switch (g.logny * 2 + (nz > 1)) {
#define CASE_B7(L) case 2 * L: y_conv_body7<L, LOGTC7, false, 1, T>(g, S.data(), Kc.data(), tw, ilog2(twN), smem.data(), b, 0, 1, nullptr, nobar, nullptr); break; \
                   case 2 * L + 1: y_conv_body7<L, LOGTC7, true, 1, T>(g, S.data(), Kc.data(), tw, ilog2(twN), smem.data(), b, 0, 1, nullptr, nobar, nullptr); break;
                CASE_B7(4) CASE_B7(5) CASE_B7(6) CASE_B7(7) CASE_B7(8) CASE_B7(9) CASE_B7(10)
            }
        } else if (b5) {
            if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body5<T, (sizeof(T) == 4 ? 2 : 1)>(g, S.data(), Kc.data(), tw, smem.data(), b, 0, 1, nullptr, nullptr);
            else y_conv_body5<T, 1>(g, S.data(), Kc.data(), tw, smem.data(), b, 0, 1, nullptr, nullptr);
        } else if (!b2) y_conv_body<T>(g, S.data(), Kh.data(), tw, smem.data(), b, 0, 1);
        else if (sizeof(T) == 4 && TC % 2 == 0) y_conv_body2<T, (sizeof(T) == 4 ? 2 : 1)>(g, S.data(), Kc.data(), tw, smem.data(), b, 0, 1);
        else y_conv_body2<T, 1>(g, S.data(), Kc.data(), tw, smem.data(), b, 0, 1);
    }
    if (b3) S.swap(S2);
    for (int b = 0; b < gridA; b++) {
        if (!a2) inv_zx_body<T>(g, S.data(), Hdt.data(), tw, (T)(1.0 / P), smem.data(), b, 0, 1);
        else switch (nz) {
#define CASE_C(NZ) case NZ: if (NZ <= 4 && g.xpad) inv_zx_body3<T, NZ, (NZ <= 4)>(g, S.data(), Hdt.data(), tw, (T)(1.0 / P), smem.data(), b, 0, 1); else inv_zx_body3<T, NZ, false>(g, S.data(), Hdt.data(), tw, (T)(1.0 / P), smem.data(), b, 0, 1); break;
            CASE_C(1) CASE_C(2) CASE_C(4) CASE_C(8) CASE_C(16) CASE_C(32)
        }
    }
    for (long i = 0; i < 3 * g.N; i++) Hd[i] = (double)Hdt[i];
}

extern "C" void emul_demag(int ver, int prec64, int nx, int ny, int nz, int G, int CH, int TC, const double* Kfull, const double* Ms,
                           const double* m, double* Hd)
{
    if (prec64) run<double>(ver, nx, ny, nz, G, CH, TC, Kfull, Ms, m, Hd);
    else run<float>(ver, nx, ny, nz, G, CH, TC, Kfull, Ms, m, Hd);
}

// local field + torque, cell by cell (terms bitmask as in LocalP)
extern "C" void emul_local(int nx, int ny, int nz, const double* par /* cex3,cdm3,cku,u3,h3,gp,agp */, int dmi, int terms,
                           const double* Ms, const double* m, const double* Hd, int torque, double* out)
{
    Geom g = make_geom(nx, ny, nz, 1, 8, 1);
    LocalP<double> lp;
    for (int a = 0; a < 3; a++) { lp.cex[a] = par[a]; lp.cdm[a] = par[3 + a]; lp.u[a] = par[7 + a]; lp.hext[a] = par[10 + a]; }
    lp.cku = par[6]; lp.gp = par[13]; lp.agp = par[14]; lp.dmi = dmi; lp.terms = terms;
    lp.ckc = 0; lp.Acell = nullptr; lp.Dcell = nullptr; lp.Hcell = nullptr; lp.Hth = nullptr; lp.stt_on = 0; lp.sl_on = 0; lp.stt_b = 0; lp.stt_w = 0;
    const long N = g.N;
    for (long q = 0; q < N; q++) {
        v3<double> res = { 0, 0, 0 };
        if (Ms[q] != 0.0) {
            int i = (int)(q % nx), j = (int)((q / nx) % ny), k = (int)(q / ((long)nx * ny));
            v3<double> mi = ld3(m, N, q), H = { 0, 0, 0 };
            if (Hd) H = ld3(Hd, N, q);
            H = local_field<double>(g, lp, m, Ms, i, j, k, q, Ms[q], mi, H);
            res = torque ? ll_torque<double>(lp, mi, H) : H;
        }
        out[q] = res.x; out[N + q] = res.y; out[2 * N + q] = res.z;
    }
}

// the same with the (f)2 parameters: cell-based A / D (nullptr = uniform), cubic constant ckc = 4Kc/mu0, per-cell H_ext
extern "C" void emul_local2(int nx, int ny, int nz, const double* par /* cex3,cdm3,cku,u3,h3,gp,agp,ckc */, int dmi, int terms,
                            const double* Ms, const double* m, const double* Acell, const double* Dcell, const double* Hcell, int torque, double* out)
{
    Geom g = make_geom(nx, ny, nz, 1, 8, 1);
    LocalP<double> lp;
    for (int a = 0; a < 3; a++) { lp.cex[a] = par[a]; lp.cdm[a] = par[3 + a]; lp.u[a] = par[7 + a]; lp.hext[a] = par[10 + a]; }
    lp.cku = par[6]; lp.gp = par[13]; lp.agp = par[14]; lp.ckc = par[15]; lp.dmi = dmi; lp.terms = terms;
    lp.Acell = Acell; lp.Dcell = Dcell; lp.Hcell = Hcell; lp.Hth = nullptr; lp.stt_on = 0; lp.sl_on = 0; lp.stt_b = 0; lp.stt_w = 0;
    const long N = g.N;
    for (long q = 0; q < N; q++) {
        v3<double> res = { 0, 0, 0 };
        if (Ms[q] != 0.0) {
            int i = (int)(q % nx), j = (int)((q / nx) % ny), k = (int)(q / ((long)nx * ny));
            v3<double> mi = ld3(m, N, q), H = { 0, 0, 0 };
            H = local_field<double>(g, lp, m, Ms, i, j, k, q, Ms[q], mi, H);
            res = torque ? ll_torque<double>(lp, mi, H) : H;
        }
        out[q] = res.x; out[N + q] = res.y; out[2 * N + q] = res.z;
    }
}
