// Step a0: the plane-wave sphere and its index maps, host code, integer arithmetic only.
// Reading R2: inclusion |n|^2 <= n2max; order ascending lexicographic in the signed triple (n_x,n_y,n_z).
// The GAMMA half sphere {0} U {first non-zero component positive} is the contiguous tail of that list starting at n = 0.
#pragma once
#include <cstdint>
#include <vector>

struct HostSphere {
    int N = 0, n2max = 0, n_max = 0, gamma = 0;
    int64_t n_full = 0, n_g = 0;              // n_g follows the mode
    std::vector<int32_t> miller;              // [n_g][3] in storage order
    std::vector<double> g2;                   // [n_g]
    // disc of (n_x, n_y) columns, lexicographic; always the FULL disc
    int n_cols = 0, nr = 0;
    std::vector<int32_t> row_off;             // [nr+1]
    // work units of the z-stick kernels: FULL: every column; GAMMA: the stored half of the columns (tail from (0,0))
    int n_units = 0;
    std::vector<int32_t> unit_off, unit_zmax; // [n_units]
};

static inline int isqrt_floor(int v) {
    int r = 0;
    while ((r + 1) * (r + 1) <= v) ++r;
    return r;
}

static inline HostSphere build_sphere(int n2max, int N, int gamma, double L) {
    HostSphere s;
    s.N = N; s.n2max = n2max; s.gamma = gamma;
    const int m = isqrt_floor(n2max);
    s.n_max = m;
    s.nr = 2 * m + 1;
    const double tpiba = 2.0 * 3.14159265358979323846264338327950288 / L;
    // full list, lexicographic
    std::vector<int32_t> full;
    s.row_off.assign(s.nr + 1, 0);
    std::vector<int32_t> col_start, col_zmax, col_nx, col_ny;   // start offset in the FULL list
    for (int nx = -m; nx <= m; ++nx) {
        s.row_off[nx + m] = (int32_t)col_start.size();
        for (int ny = -m; ny <= m; ++ny) {
            const int rem = n2max - nx * nx - ny * ny;
            if (rem < 0) continue;
            const int zm = isqrt_floor(rem);
            col_start.push_back((int32_t)(full.size() / 3));
            col_zmax.push_back(zm); col_nx.push_back(nx); col_ny.push_back(ny);
            for (int nz = -zm; nz <= zm; ++nz) { full.push_back(nx); full.push_back(ny); full.push_back(nz); }
        }
    }
    s.row_off[s.nr] = (int32_t)col_start.size();
    s.n_cols = (int)col_start.size();
    s.n_full = (int64_t)(full.size() / 3);
    int64_t first = 0;                         // storage = full[first:]
    int first_col = 0;
    if (gamma) {
        first = (s.n_full - 1) / 2;            // index of (0,0,0): the list is point-symmetric about its middle
        first_col = (s.n_cols - 1) / 2;        // column (0,0)
    }
    s.n_g = s.n_full - first;
    s.miller.assign(full.begin() + 3 * first, full.end());
    s.g2.resize(s.n_g);
    for (int64_t i = 0; i < s.n_g; ++i) {
        const int64_t a = s.miller[3 * i], b = s.miller[3 * i + 1], c = s.miller[3 * i + 2];
        s.g2[i] = tpiba * tpiba * (double)(a * a + b * b + c * c);
    }
    s.n_units = s.n_cols - first_col;
    s.unit_off.resize(s.n_units);
    s.unit_zmax.resize(s.n_units);
    for (int u = 0; u < s.n_units; ++u) {
        const int c = first_col + u;
        s.unit_zmax[u] = col_zmax[c];
        // in GAMMA mode the (0,0) stick is stored from n_z = 0 on, i.e. it starts at `first`
        int64_t off = (int64_t)col_start[c] - first;
        if (gamma && u == 0) off = 0;
        s.unit_off[u] = (int32_t)off;
    }
    return s;
}
