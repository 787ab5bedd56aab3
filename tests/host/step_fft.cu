// Host-stepped run of the FFT kernel phases (paper_2203_05623_b200/csrc/fft_kernels.cuh) for tests/test_host_stepped_fft.py:
// every phase between two barriers is a function of (tid, nthreads), so the exact device code path of K1 -> K2<K2_H> -> K3
// (local part of H: T + V_loc) is executed here thread by thread on the CPU.   usage: step_fft N n2max gamma L nvec f32 in out [nb]
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <vector>
#include "../../paper_2203_05623_b200/csrc/fft_kernels.cuh"
#include "../../paper_2203_05623_b200/csrc/gsphere.hpp"

static int g_nb = 1;         // 1 or 2: items per thread and pass of the plane-kernel phases (K2's NB)

template <typename T, int N1, int N2, bool GAMMA>
void run(HostSphere& s, int nvec, std::vector<double>& X, std::vector<double>& V, std::vector<double>& Y) {
    constexpr int N = N1 * N2, CU = 5, LC = 3;
    const int NT = 40;                                   // deliberately not a multiple of anything
    WestGeom g;
    g.N = N; g.n_max = s.n_max; g.nr = s.nr; g.n_cols = s.n_cols; g.n_units = s.n_units; g.gamma = GAMMA; g.n_g = s.n_g;
    g.row_off = s.row_off.data(); g.unit_off = s.unit_off.data(); g.unit_zmax = s.unit_zmax.data(); g.g2 = s.g2.data();
    std::vector<cx<T>> tw(2 * N);                        // the two lane-friendly orders of load_tw
    for (int i = 0; i < N; ++i) {
        const int k1 = i / N2, n2 = i % N2, j = i / N1, k1b = i % N1;
        const double a = 2 * M_PI * (n2 * k1) / N, b = 2 * M_PI * (k1b * j) / N;
        tw[i] = mk<T>((T)cos(a), (T)sin(a));
        tw[N + i] = mk<T>((T)cos(b), (T)sin(b));
    }
    g.tw = nullptr;
    const int nslots = GAMMA ? (nvec + 1) / 2 : nvec;
    VecMap vm{GAMMA ? 2 : 1, GAMMA ? 1 : 0, nvec, 0};
    std::vector<cx<T>> W((size_t)nslots * N * s.n_cols);
    using KA = K1<T, N1, N2, GAMMA, CU>; using KC = K3<T, N1, N2, GAMMA, CU>; using KB = K2<T, N1, N2, K2_H, LC>;
    std::vector<T> Vp(KB::vloc_elems(), (T)0);
    auto jof = [&](int p) { return p / N2 + N1 * (p % N2); };
    for (int pz = 0; pz < N; pz++) for (int py = 0; py < N; py++) for (int px = 0; px < N; px++)     // px = N2 k1 + k2
        Vp[KB::vloc_index(pz, py - py % LC, py % LC, px / N2, px % N2)] = (T)V[((size_t)jof(px) * N + jof(py)) * N + jof(pz)];
    std::vector<cx<T>> lines(KA::NL * KA::PITCH);
    for (int slot = 0; slot < nslots; slot++) for (int u0 = 0; u0 < s.n_units; u0 += CU) {
        for (int t = 0; t < NT; t++) KA::phaseA2(t, NT, lines.data(), tw.data(), g, vm, slot, u0, (const cx<double>*)X.data());
        for (int t = 0; t < NT; t++) KA::phaseBC(t, NT, lines.data(), g, slot, u0, W.data());
    }
    K2Args<T> a{}; a.W = W.data(); a.V = Vp.data();
    std::vector<cx<T>> S(s.nr * KB::PITCH), Xl(LC * KB::PITCH);
    for (int slot = 0; slot < nslots; slot++) for (int pz = 0; pz < N; pz++) {
        cx<T>* Wp = W.data() + ((size_t)slot * N + pz) * s.n_cols;
        for (int r0 = 0; r0 < s.nr; r0 += 4) {           // row groups, as the warps of the device kernel take them
            const int nrow = s.nr - r0 < 4 ? s.nr - r0 : 4;
            if (g_nb == 2) { for (int t = 0; t < NT; t++) KB::template yA<2>(t, NT, S.data(), tw.data(), g, Wp, r0, nrow); }
            else { for (int t = 0; t < NT; t++) KB::yA(t, NT, S.data(), tw.data(), g, Wp, r0, nrow); }
            if (g_nb == 2) { for (int t = 0; t < NT; t++) KB::template yB<2>(t, NT, S.data(), g, r0, nrow); }
            else { for (int t = 0; t < NT; t++) KB::yB(t, NT, S.data(), g, r0, nrow); }
        }
        for (int py0 = 0; py0 < N; py0 += LC) {
            if (g_nb == 2) {
                for (int t = 0; t < NT; t++) KB::template xA<2>(t, NT, S.data(), Xl.data(), tw.data(), g, py0);
                for (int t = 0; t < NT; t++) KB::template xB<2>(t, NT, Xl.data(), tw.data(), a, slot, pz, py0);
                for (int t = 0; t < NT; t++) KB::template xC<2>(t, NT, S.data(), Xl.data(), g, py0);
            } else {
                for (int t = 0; t < NT; t++) KB::xA(t, NT, S.data(), Xl.data(), tw.data(), g, py0);
                for (int t = 0; t < NT; t++) KB::xB(t, NT, Xl.data(), tw.data(), a, slot, pz, py0);
                for (int t = 0; t < NT; t++) KB::xC(t, NT, S.data(), Xl.data(), g, py0);
            }
        }
        if (g_nb == 2) {
            for (int t = 0; t < NT; t++) KB::template yC<2>(t, NT, S.data(), tw.data(), g, 0, s.nr);
            for (int t = 0; t < NT; t++) KB::template yD<2>(t, NT, S.data(), g, Wp, 0, s.nr);
        } else {
            for (int t = 0; t < NT; t++) KB::yC(t, NT, S.data(), tw.data(), g, 0, s.nr);
            for (int t = 0; t < NT; t++) KB::yD(t, NT, S.data(), g, Wp, 0, s.nr);
        }
    }
    K3Epi e; e.scale = 1.0 / ((double)N * N * N); e.kinetic = 1; e.shift = nullptr; e.omega = 0; e.X = (const cx<double>*)X.data();
    for (int slot = 0; slot < nslots; slot++) for (int u0 = 0; u0 < s.n_units; u0 += CU) {
        for (int t = 0; t < NT; t++) KC::phaseAB(t, NT, lines.data(), tw.data(), g, slot, u0, W.data());
        for (int t = 0; t < NT; t++) KC::phaseC(t, NT, lines.data(), g, vm, slot, u0, e, (cx<double>*)Y.data());
    }
}

int main(int argc, char** argv) {
    if (argc < 9) return 2;
    const int N = atoi(argv[1]), n2max = atoi(argv[2]), gamma = atoi(argv[3]);
    const double L = atof(argv[4]);
    const int nvec = atoi(argv[5]), f32 = atoi(argv[6]);
    if (argc > 9) g_nb = atoi(argv[9]);
    HostSphere s = build_sphere(n2max, N, gamma, L);
    std::vector<double> X((size_t)nvec * s.n_g * 2), Y(X.size(), 0.0), V((size_t)N * N * N);
    FILE* f = fopen(argv[7], "rb");
    if (!f || fread(X.data(), 8, X.size(), f) != X.size() || fread(V.data(), 8, V.size(), f) != V.size()) return 3;
    fclose(f);
#define GO(T, a, b) { if (gamma) run<T, a, b, true>(s, nvec, X, V, Y); else run<T, a, b, false>(s, nvec, X, V, Y); }
#define GO2(a, b) { if (f32) GO(float, a, b) else GO(double, a, b) }
    if (N == 24) GO2(4, 6) else if (N == 36) GO2(6, 6) else if (N == 48) GO2(6, 8) else if (N == 72) GO2(8, 9) else return 4;
    f = fopen(argv[8], "wb");
    fwrite(Y.data(), 8, Y.size(), f);
    fwrite(s.miller.data(), 4, s.miller.size(), f);
    fclose(f);
    return 0;
}
