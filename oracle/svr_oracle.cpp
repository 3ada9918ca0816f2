// TEST INFRASTRUCTURE - CPU oracle for the sparse-voxel tile rasterizer.
//
// A plain, slow, obviously-correct restatement of what the hot path computes, written from
// /root/reference/PAPER.md ("P:n" = line n) and the readings listed in DESIGN.md ("R#").
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
// build, load or call this file. It shares no code with paper_2511_02510_b200/csrc.
//
// Part A (fp64): one ray per pixel (eq. 1), EVERY voxel slab-tested against it, the hits
//   depth-sorted per ray, then ordered alpha compositing exactly as eqs. 2-4, w_max as
//   eq. 5, and the analytic gradient of sum(G * image) w.r.t. corner raw densities and SH
//   coefficients ("gradients from the image loss flow directly to voxel parameters").
//   "bucketed" mode restricts each ray's brute force to the voxels whose fp64 screen rectangle
//   (dilated by one pixel) touches the ray's 32x32-pixel block: same hit set, same sums.
// Part B (fp32, fixed operation order, compiled with -ffp-contract=off): the integer mechanism
//   outputs that must match bit-exactly - per-voxel pixel rectangles, per-tile direction-octant
//   masks, the sorted (tile | octant | flipped Morton) keys with voxel ids, per-(tile,octant) ranges.
//   None of this is in the paper (P:112 says only "project"); the specification is DESIGN.md B1-B4.
//
// Pins (tests/test_oracle_pins.py): alpha = 1 - exp(-sigma l) for a constant-density voxel; empty
// scene -> background; sum_k w_k + T_K = 1; chord lengths e and sqrt(3) e; K-independence for constant
// raw; exponential-density closed form at O(K^-2); SH orthonormality by quadrature; finite differences
// on <= 8-voxel scenes; storage-order invariance; key order == per-ray t_mid order; every fp64 hit has a
// list entry. PARITY UNPINNED (definitions the paper is silent on, nothing external fixes them):
// activation placement and midpoint samples (R5), per-voxel view direction / 0.5 offset / clamp (R6),
// depth definition (R7), z_near straddle rule (B1), T_min (R8).
#include <algorithm>
#include <cmath>
#include <cstdint>
#include <cstring>
#include <limits>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct OrcScene {
    int64_t n;
    int32_t sh_degree;       // 0..3
    int32_t max_level;       // Lmax for Morton codes (part B)
    double root_lo[3];
    double root_edge;
    const uint16_t* ijkl;    // [n,4] ix,iy,iz,level
    const double* raw;       // [n,8]  corner c = bx + 2 by + 4 bz
    const double* sh;        // [n,(D+1)^2,3], basis index i = l(l+1)+m
};

struct OrcCamera {
    int32_t W, H;
    float fx, fy, cx, cy;
    float R[9];              // world -> camera, row-major
    float t[3];
    float z_near;
    float bg[3];
};

}  // extern "C"

namespace {

// ------------------------------------------------------------------------------------------
// Part A: fp64 definition
// ------------------------------------------------------------------------------------------
struct Box { double lo[3]; double e; };

// R1: level-L edge = root_edge / 2^L (larger level = finer), lo = root_lo + (ix,iy,iz) e.
inline Box voxel_box(const OrcScene& s, int64_t v) {
    Box b;
    const uint16_t* q = s.ijkl + 4 * v;
    b.e = s.root_edge * std::ldexp(1.0, -(int)q[3]);
    for (int a = 0; a < 3; ++a) b.lo[a] = s.root_lo[a] + (double)q[a] * b.e;
    return b;
}

struct Ray { double o[3], d[3]; };

// R2/R3 (eq. 1): pinhole, pixel centre (x+.5, y+.5), unit direction, o = -R^T t.
inline void camera_centre(const OrcCamera& c, double o[3]) {
    for (int a = 0; a < 3; ++a)
        o[a] = -((double)c.R[0 + a] * c.t[0] + (double)c.R[3 + a] * c.t[1] + (double)c.R[6 + a] * c.t[2]);
}

inline Ray make_ray(const OrcCamera& c, int x, int y) {
    Ray r;
    camera_centre(c, r.o);
    double u = ((double)x + 0.5 - (double)c.cx) / (double)c.fx;
    double v = ((double)y + 0.5 - (double)c.cy) / (double)c.fy;
    double n2 = 0;
    for (int a = 0; a < 3; ++a) {
        r.d[a] = (double)c.R[0 + a] * u + (double)c.R[3 + a] * v + (double)c.R[6 + a];
        n2 += r.d[a] * r.d[a];
    }
    double inv = 1.0 / std::sqrt(n2);
    for (int a = 0; a < 3; ++a) r.d[a] *= inv;
    return r;
}

// R4: slab test, t >= 0, hit iff t_out - t_in > 0.
inline bool segment(const Ray& r, const Box& b, double& tin, double& tout) {
    double t0 = 0.0, t1 = std::numeric_limits<double>::infinity();
    for (int a = 0; a < 3; ++a) {
        double lo = b.lo[a], hi = b.lo[a] + b.e;
        if (r.d[a] == 0.0) {
            if (!(lo <= r.o[a] && r.o[a] < hi)) return false;
        } else {
            double ta = (lo - r.o[a]) / r.d[a], tb = (hi - r.o[a]) / r.d[a];
            t0 = std::max(t0, std::min(ta, tb));
            t1 = std::min(t1, std::max(ta, tb));
        }
    }
    tin = t0;
    tout = t1;
    return tout - tin > 0.0;
}

// R5: K midpoint samples of the trilinearly interpolated raw density, exp AFTER interpolation
// (act_mode 1 = exp at the corners, kept for documentation only). Returns tau; optionally
// d tau / d raw[c].
inline double integrate(const Ray& r, const Box& b, double tin, double tout, int K, const double* raw,
                        int act_mode, double* dtau) {
    double l = tout - tin, sum = 0.0;
    if (dtau) for (int c = 0; c < 8; ++c) dtau[c] = 0.0;
    for (int j = 0; j < K; ++j) {
        double t = tin + ((double)j + 0.5) * l / (double)K;
        double q[3];
        for (int a = 0; a < 3; ++a) {
            q[a] = (r.o[a] + t * r.d[a] - b.lo[a]) / b.e;
            q[a] = std::min(1.0, std::max(0.0, q[a]));
        }
        double Wc[8];
        for (int c = 0; c < 8; ++c) {
            double w = 1.0;
            for (int a = 0; a < 3; ++a) w *= ((c >> a) & 1) ? q[a] : 1.0 - q[a];
            Wc[c] = w;
        }
        if (act_mode == 0) {
            double rj = 0.0;
            for (int c = 0; c < 8; ++c) rj += raw[c] * Wc[c];
            double s = std::exp(rj);
            sum += s;
            if (dtau) for (int c = 0; c < 8; ++c) dtau[c] += s * Wc[c];
        } else {
            for (int c = 0; c < 8; ++c) {
                double sc = std::exp(raw[c]);
                sum += sc * Wc[c];
                if (dtau) dtau[c] += sc * Wc[c];
            }
        }
    }
    if (dtau) for (int c = 0; c < 8; ++c) dtau[c] *= l / (double)K;
    return l / (double)K * sum;
}

// R6: real spherical harmonics, no Condon-Shortley phase, index i = l(l+1)+m, (x,y,z) = unit dir.
void sh_basis(int degree, const double d[3], double* Y) {
    const double PI = 3.14159265358979323846;
    double x = d[0], y = d[1], z = d[2];
    Y[0] = 0.5 * std::sqrt(1.0 / PI);
    if (degree < 1) return;
    double c1 = std::sqrt(3.0 / (4.0 * PI));
    Y[1] = c1 * y; Y[2] = c1 * z; Y[3] = c1 * x;
    if (degree < 2) return;
    double c2 = 0.5 * std::sqrt(15.0 / PI);
    Y[4] = c2 * x * y;
    Y[5] = c2 * y * z;
    Y[6] = 0.25 * std::sqrt(5.0 / PI) * (3.0 * z * z - 1.0);
    Y[7] = c2 * x * z;
    Y[8] = 0.25 * std::sqrt(15.0 / PI) * (x * x - y * y);
    if (degree < 3) return;
    Y[9]  = 0.25 * std::sqrt(35.0 / (2.0 * PI)) * y * (3.0 * x * x - y * y);
    Y[10] = 0.5 * std::sqrt(105.0 / PI) * x * y * z;
    Y[11] = 0.25 * std::sqrt(21.0 / (2.0 * PI)) * y * (5.0 * z * z - 1.0);
    Y[12] = 0.25 * std::sqrt(7.0 / PI) * z * (5.0 * z * z - 3.0);
    Y[13] = 0.25 * std::sqrt(21.0 / (2.0 * PI)) * x * (5.0 * z * z - 1.0);
    Y[14] = 0.25 * std::sqrt(105.0 / PI) * z * (x * x - y * y);
    Y[15] = 0.25 * std::sqrt(35.0 / (2.0 * PI)) * x * (x * x - 3.0 * y * y);
}

inline void voxel_dir(const OrcScene& s, const double o[3], int64_t v, double dir[3]) {
    Box b = voxel_box(s, v);
    double n2 = 0;
    for (int a = 0; a < 3; ++a) { dir[a] = b.lo[a] + 0.5 * b.e - o[a]; n2 += dir[a] * dir[a]; }
    if (n2 == 0.0) { dir[0] = 0; dir[1] = 0; dir[2] = 1; return; }
    double inv = 1.0 / std::sqrt(n2);
    for (int a = 0; a < 3; ++a) dir[a] *= inv;
}

// R6: c_v = max(0, 0.5 + sum_i Y_i(dir_v) sh[v,i,:]), dir_v = normalize(x_v - o); one colour per
// (voxel, camera) as eq. 4 uses c_{v_k} with no ray dependence.
void voxel_rgb(const OrcScene& s, const OrcCamera& c, double* rgb, double* pre) {
    double o[3];
    camera_centre(c, o);
    int nb = (s.sh_degree + 1) * (s.sh_degree + 1);
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < s.n; ++v) {
        double dir[3], Y[16];
        voxel_dir(s, o, v, dir);
        sh_basis(s.sh_degree, dir, Y);
        for (int ch = 0; ch < 3; ++ch) {
            double acc = 0.5;
            for (int i = 0; i < nb; ++i) acc += Y[i] * s.sh[(v * nb + i) * 3 + ch];
            if (pre) pre[v * 3 + ch] = acc;
            rgb[v * 3 + ch] = std::max(0.0, acc);
        }
    }
}

struct Hit { double tmid; int64_t v; double tin, tout; };
inline bool hit_less(const Hit& a, const Hit& b) { return a.tmid < b.tmid || (a.tmid == b.tmid && a.v < b.v); }

// fp64 screen buckets for "bucketed" mode: block (bx,by) of 32x32 pixels -> voxels whose projected
// rectangle, dilated by 1 px, touches it. Voxels with a corner at Z < 1e-6 go to every block.
struct Buckets {
    int nbx = 0, nby = 0;
    std::vector<std::vector<int64_t>> cells;
    void build(const OrcScene& s, const OrcCamera& c) {
        nbx = (c.W + 31) / 32; nby = (c.H + 31) / 32;
        cells.assign((size_t)nbx * nby, {});
        for (int64_t v = 0; v < s.n; ++v) {
            Box b = voxel_box(s, v);
            double u0 = 1e300, u1 = -1e300, v0 = 1e300, v1 = -1e300, zmin = 1e300, zmax = -1e300;
            for (int k = 0; k < 8; ++k) {
                double P[3], Q[3];
                for (int a = 0; a < 3; ++a) P[a] = b.lo[a] + (((k >> a) & 1) ? b.e : 0.0);
                for (int i = 0; i < 3; ++i)
                    Q[i] = (double)c.R[3 * i] * P[0] + (double)c.R[3 * i + 1] * P[1] + (double)c.R[3 * i + 2] * P[2] + (double)c.t[i];
                zmin = std::min(zmin, Q[2]); zmax = std::max(zmax, Q[2]);
                if (Q[2] > 0) {
                    double uu = (double)c.fx * Q[0] / Q[2] + (double)c.cx, vv = (double)c.fy * Q[1] / Q[2] + (double)c.cy;
                    u0 = std::min(u0, uu); u1 = std::max(u1, uu); v0 = std::min(v0, vv); v1 = std::max(v1, vv);
                }
            }
            if (!(zmax > 0)) continue;                      // wholly behind: no ray with t >= 0 reaches it
            int bx0 = 0, bx1 = nbx - 1, by0 = 0, by1 = nby - 1;
            if (zmin >= 1e-6) {
                u0 -= 1; v0 -= 1; u1 += 1; v1 += 1;
                if (u1 < 0 || u0 >= c.W || v1 < 0 || v0 >= c.H) continue;
                bx0 = (int)std::floor(std::max(u0, 0.0)) / 32; bx1 = (int)std::floor(std::min(u1, c.W - 1.0)) / 32;
                by0 = (int)std::floor(std::max(v0, 0.0)) / 32; by1 = (int)std::floor(std::min(v1, c.H - 1.0)) / 32;
            }
            for (int by = by0; by <= by1; ++by)
                for (int bx = bx0; bx <= bx1; ++bx) cells[(size_t)by * nbx + bx].push_back(v);
        }
    }
};

inline void collect_hits(const OrcScene& s, const Ray& r, const std::vector<int64_t>* cand, std::vector<Hit>& hits) {
    hits.clear();
    int64_t m = cand ? (int64_t)cand->size() : s.n;
    for (int64_t i = 0; i < m; ++i) {
        int64_t v = cand ? (*cand)[i] : i;
        Box b = voxel_box(s, v);
        double tin, tout;
        if (segment(r, b, tin, tout)) hits.push_back({0.5 * (tin + tout), v, tin, tout});
    }
    std::sort(hits.begin(), hits.end(), hit_less);            // R7: front-to-back by t_mid
}

inline void atomic_max_double(double* addr, double val) {      // non-negative doubles only
    uint64_t* p = reinterpret_cast<uint64_t*>(addr);
    uint64_t nv;
    std::memcpy(&nv, &val, 8);
    uint64_t old = __atomic_load_n(p, __ATOMIC_RELAXED);
    while (old < nv && !__atomic_compare_exchange_n(p, &old, nv, true, __ATOMIC_RELAXED, __ATOMIC_RELAXED)) {}
}

inline void ray_xy(const OrcCamera& c, const int32_t* xy, int64_t i, int& x, int& y) {
    if (xy) { x = xy[2 * i]; y = xy[2 * i + 1]; }
    else { x = (int)(i % c.W); y = (int)(i / c.W); }
}

// ------------------------------------------------------------------------------------------
// Part B: fp32 binning specification (B1-B4). Every operation is a separate, individually
// rounded binary32 operation in the written order; built with -ffp-contract=off.
// ------------------------------------------------------------------------------------------
struct RectU16 { uint16_t x0, y0, x1, y1; };

inline RectU16 bin_rect(const OrcScene& s, const OrcCamera& c, int64_t v) {
    const RectU16 culled = {0xFFFF, 0xFFFF, 0, 0};
    const uint16_t* q = s.ijkl + 4 * v;
    float e = std::ldexp((float)s.root_edge, -(int)q[3]);
    float lo[3], hi[3];
    for (int a = 0; a < 3; ++a) {
        float off = (float)q[a] * e;
        lo[a] = (float)s.root_lo[a] + off;
        hi[a] = lo[a] + e;
    }
    float X[8], Y[8], Z[8];
    float zmin = 0, zmax = 0;
    for (int k = 0; k < 8; ++k) {
        float Px = (k & 1) ? hi[0] : lo[0], Py = (k & 2) ? hi[1] : lo[1], Pz = (k & 4) ? hi[2] : lo[2];
        float m0, m1, m2, acc;
        m0 = c.R[0] * Px; m1 = c.R[1] * Py; m2 = c.R[2] * Pz; acc = m0 + m1; acc = acc + m2; X[k] = acc + c.t[0];
        m0 = c.R[3] * Px; m1 = c.R[4] * Py; m2 = c.R[5] * Pz; acc = m0 + m1; acc = acc + m2; Y[k] = acc + c.t[1];
        m0 = c.R[6] * Px; m1 = c.R[7] * Py; m2 = c.R[8] * Pz; acc = m0 + m1; acc = acc + m2; Z[k] = acc + c.t[2];
        if (k == 0) { zmin = zmax = Z[k]; }
        else { zmin = std::fmin(zmin, Z[k]); zmax = std::fmax(zmax, Z[k]); }
    }
    if (!(zmax > 0.0f)) return culled;                        // wholly behind the camera plane
    float Wf = (float)c.W, Hf = (float)c.H;
    if (zmin < c.z_near) {
        // straddles the near plane: cull only if one image-side half-space excludes all 8 corners
        // (homogeneous test, valid whatever the sign of Z); otherwise the whole image.
        float cxw = c.cx - Wf, cyh = c.cy - Hf;
        bool allL = true, allR = true, allT = true, allB = true;
        for (int k = 0; k < 8; ++k) {
            float a0 = c.fx * X[k], a1, h;
            a1 = c.cx * Z[k]; h = a0 + a1; allL = allL && (h < 0.0f);
            a1 = cxw * Z[k];  h = a0 + a1; allR = allR && (h >= 0.0f);
            float b0 = c.fy * Y[k];
            a1 = c.cy * Z[k]; h = b0 + a1; allT = allT && (h < 0.0f);
            a1 = cyh * Z[k];  h = b0 + a1; allB = allB && (h >= 0.0f);
        }
        if (allL || allR || allT || allB) return culled;
        return {0, 0, (uint16_t)(c.W - 1), (uint16_t)(c.H - 1)};
    }
    float u0 = 0, u1 = 0, v0 = 0, v1 = 0;
    for (int k = 0; k < 8; ++k) {
        float xz = X[k] / Z[k], yz = Y[k] / Z[k];
        float u = c.fx * xz; u = u + c.cx;
        float w = c.fy * yz; w = w + c.cy;
        if (k == 0) { u0 = u1 = u; v0 = v1 = w; }
        else { u0 = std::fmin(u0, u); u1 = std::fmax(u1, u); v0 = std::fmin(v0, w); v1 = std::fmax(v1, w); }
    }
    if (u1 < 0.0f || u0 >= Wf || v1 < 0.0f || v0 >= Hf) return culled;
    RectU16 r;
    r.x0 = (uint16_t)(int)std::floor(std::fmax(u0, 0.0f));
    r.x1 = (uint16_t)(int)std::floor(std::fmin(u1, Wf - 1.0f));
    r.y0 = (uint16_t)(int)std::floor(std::fmax(v0, 0.0f));
    r.y1 = (uint16_t)(int)std::floor(std::fmin(v1, Hf - 1.0f));
    return r;
}

inline int pixel_octant(const OrcCamera& c, int x, int y) {
    float u = ((float)x + 0.5f); u = u - c.cx; u = u / c.fx;
    float v = ((float)y + 0.5f); v = v - c.cy; v = v / c.fy;
    int s = 0;
    for (int a = 0; a < 3; ++a) {
        float m0 = c.R[0 + a] * u, m1 = c.R[3 + a] * v;
        float d = m0 + m1; d = d + c.R[6 + a];
        if (d < 0.0f) s |= 1 << a;
    }
    return s;
}

inline uint64_t morton3(uint32_t x, uint32_t y, uint32_t z, int bits) {
    uint64_t code = 0;
    for (int b = 0; b < bits; ++b) {
        code |= (uint64_t)((x >> b) & 1) << (3 * b);
        code |= (uint64_t)((y >> b) & 1) << (3 * b + 1);
        code |= (uint64_t)((z >> b) & 1) << (3 * b + 2);
    }
    return code;
}

}  // namespace

extern "C" {

int orc_num_threads() {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void orc_sh_basis(int degree, const double* dir, double* Y) { sh_basis(degree, dir, Y); }

void orc_voxel_rgb(const OrcScene* s, const OrcCamera* c, double* rgb, double* pre) { voxel_rgb(*s, *c, rgb, pre); }

void orc_ray(const OrcCamera* c, int x, int y, double* o, double* d) {
    Ray r = make_ray(*c, x, y);
    for (int a = 0; a < 3; ++a) { o[a] = r.o[a]; d[a] = r.d[a]; }
}

// One ray, every voxel: the sorted hit list with per-hit segment, tau, alpha-composited weight.
// Returns the number of hits (fills at most max_hits).
int64_t orc_ray_dump(const OrcScene* s, const OrcCamera* c, int K, int act_mode, int x, int y, int64_t max_hits,
                     int64_t* vox, double* tin, double* tout, double* tau, double* w, double* T_final) {
    Ray r = make_ray(*c, x, y);
    std::vector<Hit> hits;
    collect_hits(*s, r, nullptr, hits);
    double T = 1.0;
    for (size_t k = 0; k < hits.size(); ++k) {
        Box b = voxel_box(*s, hits[k].v);
        double tk = integrate(r, b, hits[k].tin, hits[k].tout, K, s->raw + 8 * hits[k].v, act_mode, nullptr);
        double alpha = -std::expm1(-tk);
        if ((int64_t)k < max_hits) {
            vox[k] = hits[k].v; tin[k] = hits[k].tin; tout[k] = hits[k].tout; tau[k] = tk; w[k] = T * alpha;
        }
        T *= std::exp(-tk);
    }
    if (T_final) *T_final = T;
    return (int64_t)hits.size();
}

// Forward (eqs. 2-5). rays: xy = NULL -> all W*H pixels row-major, else n_rays (x,y) pairs.
// mode 0 = pure (all voxels per ray), 1 = bucketed. image[n_rays,3], depth, T_final [n_rays];
// w_max[n] is max-accumulated in place (caller zeroes); n_hits[n_rays] optional.
void orc_render(const OrcScene* sp, const OrcCamera* cp, int K, int act_mode, int mode, int64_t n_rays,
                const int32_t* xy, double* image, double* depth, double* T_final, double* w_max, int32_t* n_hits) {
    const OrcScene& s = *sp; const OrcCamera& c = *cp;
    std::vector<double> rgb((size_t)s.n * 3);
    voxel_rgb(s, c, rgb.data(), nullptr);
    Buckets bk;
    if (mode == 1) bk.build(s, c);
#pragma omp parallel
    {
        std::vector<Hit> hits;
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n_rays; ++i) {
            int x, y;
            ray_xy(c, xy, i, x, y);
            Ray r = make_ray(c, x, y);
            collect_hits(s, r, mode == 1 ? &bk.cells[(size_t)(y / 32) * bk.nbx + x / 32] : nullptr, hits);
            double T = 1.0, C[3] = {0, 0, 0}, D = 0.0;
            for (const Hit& h : hits) {
                Box b = voxel_box(s, h.v);
                double tau = integrate(r, b, h.tin, h.tout, K, s.raw + 8 * h.v, act_mode, nullptr);
                double alpha = -std::expm1(-tau);
                double w = T * alpha;                               // eq. 2
                for (int ch = 0; ch < 3; ++ch) C[ch] += w * rgb[h.v * 3 + ch];   // eq. 4
                D += w * h.tmid;
                if (w_max) atomic_max_double(&w_max[h.v], w);       // eq. 5
                T *= std::exp(-tau);                                // eq. 3 (1 - alpha = exp(-tau))
            }
            for (int ch = 0; ch < 3; ++ch) image[i * 3 + ch] = C[ch] + T * (double)c.bg[ch];   // R7 background
            if (depth) depth[i] = D;
            if (T_final) T_final[i] = T;
            if (n_hits) n_hits[i] = (int32_t)hits.size();
        }
    }
}

// Backward of L = sum(G * image) + sum(GD * depth) + sum(GT * T_final): grad_raw[n,8] and grad_sh[n,(D+1)^2,3]
// accumulate (+=). GD, GT (one value per ray) may be NULL. With D = sum_k w_k t_mid,k and T_K = prod_k exp(-tau_k)
// (reading R7; geometry carries no gradient, so t_mid is a constant):
//   dD/dtau_k = T_k t_mid,k - sum_{j>k} w_j t_mid,j,   dT_K/dtau_k = -T_K   (NEXT-3, heads for the depth / transmittance terms of eq. 17).
void orc_backward_heads(const OrcScene* sp, const OrcCamera* cp, int K, int act_mode, int mode, int64_t n_rays,
                        const int32_t* xy, const double* G, const double* GD, const double* GT, double* grad_raw, double* grad_sh) {
    const OrcScene& s = *sp; const OrcCamera& c = *cp;
    int nb = (s.sh_degree + 1) * (s.sh_degree + 1);
    std::vector<double> rgb((size_t)s.n * 3), pre((size_t)s.n * 3), grgb((size_t)s.n * 3, 0.0);
    voxel_rgb(s, c, rgb.data(), pre.data());
    Buckets bk;
    if (mode == 1) bk.build(s, c);
#pragma omp parallel
    {
        std::vector<Hit> hits;
        std::vector<double> tau, wk, Tk, dtau;
#pragma omp for schedule(dynamic, 16)
        for (int64_t i = 0; i < n_rays; ++i) {
            int x, y;
            ray_xy(c, xy, i, x, y);
            Ray r = make_ray(c, x, y);
            collect_hits(s, r, mode == 1 ? &bk.cells[(size_t)(y / 32) * bk.nbx + x / 32] : nullptr, hits);
            size_t n = hits.size();
            tau.resize(n); wk.resize(n); Tk.resize(n); dtau.resize(8 * n);
            double T = 1.0;
            for (size_t k = 0; k < n; ++k) {
                Box b = voxel_box(s, hits[k].v);
                tau[k] = integrate(r, b, hits[k].tin, hits[k].tout, K, s.raw + 8 * hits[k].v, act_mode, &dtau[8 * k]);
                wk[k] = T * -std::expm1(-tau[k]);
                T *= std::exp(-tau[k]);
                Tk[k] = T;
            }
            const double* g = G + 3 * i;
            const double gd = GD ? GD[i] : 0.0, gt = GT ? GT[i] : 0.0;
            double S[3];                                       // suffix colour S_k = sum_{j>k} w_j c_j + T_K bg
            for (int ch = 0; ch < 3; ++ch) S[ch] = T * (double)c.bg[ch];
            double SD = 0.0;                                   // suffix depth sum_{j>k} w_j t_mid,j
            const double TK = T;
            for (size_t kk = n; kk-- > 0;) {
                int64_t v = hits[kk].v;
                const double tmid = hits[kk].tmid;
                double dL_dtau = gd * (Tk[kk] * tmid - SD) - gt * TK;   // d alpha / d tau = 1 - alpha  =>  G.(T_k c_k - S_k)
                SD += wk[kk] * tmid;
                for (int ch = 0; ch < 3; ++ch) dL_dtau += g[ch] * (Tk[kk] * rgb[v * 3 + ch] - S[ch]);
                for (int cc = 0; cc < 8; ++cc) {
                    double add = dL_dtau * dtau[8 * kk + cc];
#pragma omp atomic
                    grad_raw[v * 8 + cc] += add;
                }
                for (int ch = 0; ch < 3; ++ch) {
                    double add = wk[kk] * g[ch];
#pragma omp atomic
                    grgb[v * 3 + ch] += add;
                    S[ch] += wk[kk] * rgb[v * 3 + ch];
                }
            }
        }
    }
    double o[3];
    camera_centre(c, o);
#pragma omp parallel for schedule(static)
    for (int64_t v = 0; v < s.n; ++v) {
        if (grgb[v * 3] == 0.0 && grgb[v * 3 + 1] == 0.0 && grgb[v * 3 + 2] == 0.0) continue;
        double dir[3], Y[16];
        voxel_dir(s, o, v, dir);
        sh_basis(s.sh_degree, dir, Y);
        for (int ch = 0; ch < 3; ++ch) {
            if (!(pre[v * 3 + ch] > 0.0)) continue;            // zero sub-gradient at the clamp
            for (int i = 0; i < nb; ++i) grad_sh[(v * nb + i) * 3 + ch] += Y[i] * grgb[v * 3 + ch];
        }
    }
}

void orc_backward(const OrcScene* sp, const OrcCamera* cp, int K, int act_mode, int mode, int64_t n_rays,
                  const int32_t* xy, const double* G, double* grad_raw, double* grad_sh) {
    orc_backward_heads(sp, cp, K, act_mode, mode, n_rays, xy, G, nullptr, nullptr, grad_raw, grad_sh);
}

// ---- part B ----
// rects[n,4] = x0,y0,x1,y1 (pixels, inclusive; culled = 65535,65535,0,0); tile_masks[n_tiles] = set of
// direction octants among the tile's pixels; returns the number of list entries E.
int64_t orc_bin_rects(const OrcScene* sp, const OrcCamera* cp, uint16_t* rects, uint8_t* tile_masks) {
    const OrcScene& s = *sp; const OrcCamera& c = *cp;
    int tx = (c.W + 15) / 16, ty = (c.H + 15) / 16;
    std::memset(tile_masks, 0, (size_t)tx * ty);
    for (int y = 0; y < c.H; ++y)
        for (int x = 0; x < c.W; ++x) tile_masks[(size_t)(y >> 4) * tx + (x >> 4)] |= (uint8_t)(1u << pixel_octant(c, x, y));
    int64_t E = 0;
    for (int64_t v = 0; v < s.n; ++v) {
        RectU16 r = bin_rect(s, c, v);
        rects[4 * v] = r.x0; rects[4 * v + 1] = r.y0; rects[4 * v + 2] = r.x1; rects[4 * v + 3] = r.y1;
        if (r.x0 > r.x1) continue;
        for (int j = r.y0 >> 4; j <= (r.y1 >> 4); ++j)
            for (int i = r.x0 >> 4; i <= (r.x1 >> 4); ++i) E += __builtin_popcount(tile_masks[(size_t)j * tx + i]);
    }
    return E;
}

int orc_pixel_octant(const OrcCamera* c, int x, int y) { return pixel_octant(*c, x, y); }

// keys[E], vals[E] sorted ascending by key; ranges[n_tiles*8*2] = [start,end) per (tile, octant), (0,0) if empty.
void orc_bin_lists(const OrcScene* sp, const OrcCamera* cp, const uint16_t* rects, const uint8_t* tile_masks,
                   uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
    const OrcScene& s = *sp; const OrcCamera& c = *cp;
    int tx = (c.W + 15) / 16, ty = (c.H + 15) / 16;
    int Lm = s.max_level;
    uint64_t xmask = 0;
    for (int b = 0; b < Lm; ++b) xmask |= (uint64_t)1 << (3 * b);
    std::vector<std::pair<uint64_t, uint32_t>> ent;
    for (int64_t v = 0; v < s.n; ++v) {
        const uint16_t* r = rects + 4 * v;
        if (r[0] > r[2]) continue;
        const uint16_t* q = s.ijkl + 4 * v;
        int sh = Lm - (int)q[3];
        uint64_t code = morton3((uint32_t)q[0] << sh, (uint32_t)q[1] << sh, (uint32_t)q[2] << sh, Lm);
        for (int j = r[1] >> 4; j <= (r[3] >> 4); ++j)
            for (int i = r[0] >> 4; i <= (r[2] >> 4); ++i) {
                uint64_t tile = (uint64_t)j * tx + i;
                uint8_t m = tile_masks[tile];
                for (int o = 0; o < 8; ++o) {
                    if (!((m >> o) & 1)) continue;
                    uint64_t flip = ((o & 1) ? xmask : 0) | ((o & 2) ? xmask << 1 : 0) | ((o & 4) ? xmask << 2 : 0);
                    uint64_t key = (tile << (3 + 3 * Lm)) | ((uint64_t)o << (3 * Lm)) | (code ^ flip);
                    ent.emplace_back(key, (uint32_t)v);
                }
            }
    }
    std::sort(ent.begin(), ent.end());
    std::memset(ranges, 0, sizeof(uint32_t) * (size_t)tx * ty * 16);
    for (size_t i = 0; i < ent.size(); ++i) {
        keys[i] = ent[i].first; vals[i] = ent[i].second;
        uint64_t p = ent[i].first >> (3 * Lm);
        if (i == 0 || (ent[i - 1].first >> (3 * Lm)) != p) ranges[2 * p] = (uint32_t)i;
        if (i + 1 == ent.size() || (ent[i + 1].first >> (3 * Lm)) != p) ranges[2 * p + 1] = (uint32_t)(i + 1);
    }
}

}  // extern "C"
