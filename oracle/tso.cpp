// oracle/tso.cpp -- CPU ORACLE (test infrastructure, NOT the product; see oracle/tso.h).
//
// Plain, slow, single-threaded restatement of the Triangle Splatting SLAM rasteriser:
//   Eq. 1   v_I = pi(T_CW v_W)                         -> project()
//   Eq. 2   phi(p) = max_i L_i(p), outward unit normals -> face_setup(), eval()
//   Eq. 3   I(p) = ReLU(phi(p)/phi(s))^sigma            -> eval()
//   :82                      barycentric vertex colour, mean vertex opacity
//   Eq. 4 front-to-back compositing in depth order    -> render_fwd()
//   Eq. 5-7 analytic se(3) pose Jacobian              -> project_bwd()
//   Eq. 12 rendered normal map                        -> face_normal(), render_fwd/bwd(nrm)
// Step names F1..F8 / B1..B9 and readings S1..S28 / N1..N11 refer to DESIGN.md section 2 (pins: section 3).
// Build: g++ -std=c++17 -O2 -ffp-contract=off (no implicit FMA contraction; the float32
// projection uses explicit std::fma where N1..N3 say so).
#include "tso.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <vector>

namespace {

template <class T>
struct Cam {
    int W, H;
    T fx, fy, cx, cy, znear;
    explicit Cam(const tso_camera* c)
        : W(c->width), H(c->height), fx((T)c->fx), fy((T)c->fy), cx((T)c->cx), cy((T)c->cy), znear((T)c->znear) {}
};

inline int vid(const int32_t* faces, int m, int k) { return faces ? faces[3 * m + k] : 3 * m + k; }

template <class T> inline T third();
template <> inline float third<float>() { return 1.0f / 3.0f; }
template <> inline double third<double>() { return 1.0 / 3.0; }

// N3: signed doubled area of the screen triangle, S = fma(a, b, -(c*d)).
template <class T>
inline T signed_area(const T u[3], const T v[3]) {
    T a = u[1] - u[0], b = v[2] - v[0], c = v[1] - v[0], d = u[2] - u[0];
    T cd = c * d;
    return std::fma(a, b, -cd);
}

// ---------------------------------------------------------------------------------- F1..F6
// S31 (tight binning): does the triangle meet the box of pixel centres [bx0,bx1] x [by0,by1]?
// For each edge k (from q_{k+1} to q_{k+2}) the un-normalised outward edge function
//     E_k(p) = s (ey (px - ua) - ex (py - va)),   s = sign(S),
// is taken at the corner of the box where it is smallest; the box is left out iff some E_k there exceeds
// 2^-10 (|ex| + |ey|), i.e. every pixel of the box is at least ~1e-3 px OUTSIDE edge k: none of them can pass the hit
// rule x > 0.  Conservative (the separating axes of the box itself are covered by the rect); fixed operation order, so
// that two float32 implementations agree bit for bit.
template <class T>
bool tile_overlaps(const T* u, const T* v, int bx0, int by0, int bx1, int by1) {
    const T a = u[1] - u[0], b = v[2] - v[0], c = v[1] - v[0], d = u[2] - u[0];
    const T S = std::fma(a, b, -(c * d));
    const T s = S > 0 ? (T)1 : (T)-1;
    for (int k = 0; k < 3; ++k) {
        const int ia = (k + 1) % 3, ib = (k + 2) % 3;
        const T ex = u[ib] - u[ia], ey = v[ib] - v[ia];
        const T sx = s * ey, sy = -(s * ex);
        const T px = sx > 0 ? (T)bx0 : (T)bx1, py = sy > 0 ? (T)by0 : (T)by1;
        const T dx = px - u[ia], dy = py - v[ia];
        const T E = std::fma(sx, dx, sy * dy);
        const T margin = (T)0.0009765625 * (std::fabs(ex) + std::fabs(ey));
        if (E > margin) return false;
    }
    return true;
}

// tiles of the rect that the face is binned into: all of them, or (tight) those its triangle meets
template <class T>
bool tile_included(bool tight, const T* u, const T* v, const int16_t* rc, int tx, int ty) {
    if (!tight) return true;
    const int bx0 = std::max((int)rc[0], tx * 16), bx1 = std::min((int)rc[2], tx * 16 + 15);
    const int by0 = std::max((int)rc[1], ty * 16), by1 = std::min((int)rc[3], ty * 16 + 15);
    return tile_overlaps<T>(u, v, bx0, by0, bx1, by1);
}

template <class T>
int64_t project(const T* pos, const int32_t* faces, int32_t M, const T* Tcw, const tso_camera* cam_,
                const tso_params* prm, uint8_t* visible, int16_t* rect, uint32_t* depth_key,
                uint32_t* tiles_touched, T* scr, T* Q, T* zbar) {
    const Cam<T> cam(cam_);
    const T eps_area = (T)prm->eps_area;
    const T area_max = (T)1e10;
    int64_t nvis = 0;
    for (int m = 0; m < M; ++m) {
        visible[m] = 0;
        tiles_touched[m] = 0;
        depth_key[m] = 0;
        zbar[m] = 0;
        for (int j = 0; j < 4; ++j) rect[4 * m + j] = 0;
        for (int j = 0; j < 9; ++j) scr[9 * m + j] = 0, Q[9 * m + j] = 0;
        T X[3], Y[3], Z[3], u[3], v[3], w[3];
        for (int k = 0; k < 3; ++k) {
            const T* p = pos + 3 * (int64_t)vid(faces, m, k);
            // F1 / N1: Q = R p + t, innermost term first.
            X[k] = std::fma(Tcw[0], p[0], std::fma(Tcw[1], p[1], std::fma(Tcw[2], p[2], Tcw[3])));
            Y[k] = std::fma(Tcw[4], p[0], std::fma(Tcw[5], p[1], std::fma(Tcw[6], p[2], Tcw[7])));
            Z[k] = std::fma(Tcw[8], p[0], std::fma(Tcw[9], p[1], std::fma(Tcw[10], p[2], Tcw[11])));
        }
        // F2: near cull, written so NaN culls.
        if (!(Z[0] > cam.znear) || !(Z[1] > cam.znear) || !(Z[2] > cam.znear)) continue;
        for (int k = 0; k < 3; ++k) {
            // F3 / N2: w = 1/Z (IEEE), X*w rounded separately, then one fma.
            w[k] = (T)1 / Z[k];
            T xw = X[k] * w[k], yw = Y[k] * w[k];
            u[k] = std::fma(cam.fx, xw, cam.cx);
            v[k] = std::fma(cam.fy, yw, cam.cy);
        }
        // F4 / N3: degenerate cull.
        T S = signed_area(u, v);
        T aS = std::fabs(S);
        if (!(aS > eps_area) || !(aS < area_max)) continue;
        // F5 / N4: integer pixel centres inside the vertex AABB, clipped to the image.
        T umin = std::fmin(u[0], std::fmin(u[1], u[2])), umax = std::fmax(u[0], std::fmax(u[1], u[2]));
        T vmin = std::fmin(v[0], std::fmin(v[1], v[2])), vmax = std::fmax(v[0], std::fmax(v[1], v[2]));
        int x0 = (int)std::fmin(std::fmax(std::ceil(umin), (T)0), (T)cam.W);
        int x1 = (int)std::fmin(std::fmax(std::floor(umax), (T)-1), (T)(cam.W - 1));
        int y0 = (int)std::fmin(std::fmax(std::ceil(vmin), (T)0), (T)cam.H);
        int y1 = (int)std::fmin(std::fmax(std::floor(vmax), (T)-1), (T)(cam.H - 1));
        if (x0 > x1 || y0 > y1) continue;
        // F6 / N5: depth key = bits of the float32 mean camera depth.
        T zb = ((Z[0] + Z[1]) + Z[2]) * third<T>();
        float zf = (float)zb;
        uint32_t bits;
        std::memcpy(&bits, &zf, 4);
        visible[m] = 1;
        rect[4 * m + 0] = (int16_t)x0, rect[4 * m + 1] = (int16_t)y0;
        rect[4 * m + 2] = (int16_t)x1, rect[4 * m + 3] = (int16_t)y1;
        depth_key[m] = bits;
        zbar[m] = zb;
        {
            uint32_t nt = 0;
            const int16_t* rc = rect + 4 * (int64_t)m;
            for (int ty = y0 >> 4; ty <= (y1 >> 4); ++ty)
                for (int tx = x0 >> 4; tx <= (x1 >> 4); ++tx) nt += tile_included<T>(prm->tight_binning != 0, u, v, rc, tx, ty) ? 1u : 0u;
            tiles_touched[m] = nt;
        }
        for (int k = 0; k < 3; ++k) {
            scr[9 * m + 3 * k + 0] = u[k], scr[9 * m + 3 * k + 1] = v[k], scr[9 * m + 3 * k + 2] = w[k];
            Q[9 * m + 3 * k + 0] = X[k], Q[9 * m + 3 * k + 1] = Y[k], Q[9 * m + 3 * k + 2] = Z[k];
        }
        ++nvis;
    }
    return nvis;
}

// ---------------------------------------------------------------------------------- F7
template <class T>
struct Face {
    T qx[3], qy[3], w[3];   // screen vertices and inverse depths
    T nx[3], ny[3];         // outward unit normal of edge k (opposite vertex k)
    T ell[3], h[3];         // edge length, altitude of vertex k
    T r, absS, sumell, s;   // inradius = -phi(s), |S|, perimeter, sign of S
    T obar;                 // face opacity = mean of vertex opacities (:82), or their minimum (ablation, :433)
    int kmin;               // min mode: the vertex the opacity gradient goes to (lowest index among equal minima)
    T col[3][3];            // vertex colours
    int x0, y0, x1, y1;
};

template <class T>
void face_setup(Face<T>& f, const T* scr9, const int16_t* rc, const T* color, const T* opacity, const int32_t* faces,
                int m, bool min_op) {
    for (int k = 0; k < 3; ++k) f.qx[k] = scr9[3 * k], f.qy[k] = scr9[3 * k + 1], f.w[k] = scr9[3 * k + 2];
    T S = signed_area(f.qx, f.qy);
    T s = S > 0 ? (T)1 : (T)-1;
    f.s = s;
    f.absS = std::fabs(S);
    f.sumell = 0;
    for (int k = 0; k < 3; ++k) {
        int a = (k + 1) % 3, b = (k + 2) % 3;   // edge k runs from q_{k+1} to q_{k+2}
        T ex = f.qx[b] - f.qx[a], ey = f.qy[b] - f.qy[a];
        f.ell[k] = std::sqrt(ex * ex + ey * ey);
        f.nx[k] = s * ey / f.ell[k];
        f.ny[k] = -s * ex / f.ell[k];
        f.h[k] = f.absS / f.ell[k];
        f.sumell += f.ell[k];
    }
    f.r = f.absS / f.sumell;
    T osum = 0;
    for (int k = 0; k < 3; ++k) {
        int v = vid(faces, m, k);
        osum += opacity[v];
        for (int c = 0; c < 3; ++c) f.col[k][c] = color[3 * (int64_t)v + c];
    }
    f.obar = osum / (T)3;
    f.kmin = -1;
    if (min_op) {
        // "the minimum operator ... routes gradients solely to the vertex with the lowest opacity"
        f.kmin = 0;
        for (int k = 1; k < 3; ++k)
            if (opacity[vid(faces, m, k)] < opacity[vid(faces, m, f.kmin)]) f.kmin = k;
        f.obar = opacity[vid(faces, m, f.kmin)];
    }
    f.x0 = rc[0], f.y0 = rc[1], f.x1 = rc[2], f.y1 = rc[3];
}

// ---------------------------------------------------------------------------------- F8.1-4
template <class T>
struct Hit {
    T L[3], x, I, alpha, b[3], om[3], Om, lam[3], z, c[3];
    int kstar;
};

// returns 0 = no contribution, 1 = contributes.  *amb set if the alpha_min decision is within amb_tol.
template <class T>
inline int eval(const Face<T>& f, T px, T py, T sigma, T alpha_min, T amb_tol, Hit<T>& h, bool* amb) {
    for (int k = 0; k < 3; ++k) {
        // Eq. 2: L_k(p) = n_k . (p - q_{k+1}) = -s * cross(e_k, p - q_{k+1}) / ell_k, evaluated relative to a vertex
        // (S6).  The cross product is formed with the compensated 2x2 determinant (one fma recovers the rounding
        // error of the first product), so L_k keeps its RELATIVE accuracy next to the edge, where sigma < 1 makes
        // dI/dx = sigma x^(sigma-1) large (N6).
        int a = (k + 1) % 3, b = (k + 2) % 3;
        const T ex = f.qx[b] - f.qx[a], ey = f.qy[b] - f.qy[a], dx = px - f.qx[a], dy = py - f.qy[a];
        const T w = ey * dx, e = std::fma(ey, dx, -w), g = std::fma(ex, dy, -w);
        h.L[k] = -f.s * (g - e) / f.ell[k];
    }
    h.kstar = 0;
    T phi = h.L[0];
    for (int k = 1; k < 3; ++k)
        if (h.L[k] > phi) phi = h.L[k], h.kstar = k;
    h.x = -phi / f.r;                       // phi(p)/phi(s), phi(s) = -r
    if (!(h.x > 0)) return 0;               // ReLU (Eq. 3)
    h.I = std::pow(h.x, sigma);
    h.alpha = f.obar * h.I;
    if (amb && amb_tol > 0 && alpha_min > 0 && std::fabs(h.alpha - alpha_min) <= amb_tol * alpha_min) *amb = true;
    if (h.alpha < alpha_min) return 0;      // S7
    for (int k = 0; k < 3; ++k) {
        h.b[k] = -h.L[k] / f.h[k];          // screen-space barycentrics
        h.om[k] = h.b[k] * f.w[k];          // perspective correction (S10)
    }
    h.Om = (h.om[0] + h.om[1]) + h.om[2];
    h.z = (T)1 / h.Om;
    for (int k = 0; k < 3; ++k) h.lam[k] = h.om[k] / h.Om;
    for (int c = 0; c < 3; ++c) h.c[c] = h.lam[0] * f.col[0][c] + h.lam[1] * f.col[1][c] + h.lam[2] * f.col[2][c];
    return 1;
}

template <class T>
struct Lists {
    const uint32_t* list;
    int64_t n_list;
    const uint32_t* ranges;   // NULL = brute
    int tiles_x;
    inline void span(int x, int y, int64_t& b, int64_t& e) const {
        if (!ranges) { b = 0, e = n_list; return; }
        int t = (y >> 4) * tiles_x + (x >> 4);
        b = ranges[2 * t], e = ranges[2 * t + 1];
    }
};

// set-up every visible face once (the per-face constants do not depend on the pixel)
// S32: window smoothness of face m: the per-face array of tso_params (Triangle Splatting's learnable sigma)
// if there is one, else the global constant the paper uses
template <class T>
inline T face_sigma(const tso_params* prm, uint32_t m) {
    return prm->face_sigma ? ((const T*)prm->face_sigma)[m] : (T)prm->sigma;
}

template <class T>
std::vector<Face<T>> setup_all(const T* color, const T* opacity, const int32_t* faces, int32_t M,
                               const uint8_t* visible, const int16_t* rect, const T* scr, bool min_op) {
    std::vector<Face<T>> F((size_t)M);
    for (int m = 0; m < M; ++m)
        if (visible[m]) face_setup(F[m], scr + 9 * (int64_t)m, rect + 4 * (int64_t)m, color, opacity, faces, m, min_op);
    return F;
}

// ---------------------------------------------------------------------------------- F8.5-6
template <class T>
void render_fwd(const T* color, const T* opacity, const int32_t* faces, int32_t M, const tso_camera* cam_,
                const tso_params* prm, const uint8_t* visible, const int16_t* rect, const T* scr,
                const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges, T* oc, T* od, T* oa,
                uint32_t* n_contrib, uint8_t* ambig, uint64_t* sig, uint64_t* counters, const T* nrm = nullptr,
                T* on = nullptr, T* on_top = nullptr) {
    const Cam<T> cam(cam_);
    const int W = cam.W, H = cam.H;
    const T sigma = (T)prm->sigma, amin = (T)prm->alpha_min, tmin = (T)prm->t_min, atol = (T)prm->amb_tol;
    std::vector<Face<T>> F = setup_all(color, opacity, faces, M, visible, rect, scr, prm->min_opacity != 0);
    Lists<T> LS{list, n_list, tile_ranges, (W + 15) / 16};
    uint64_t n_visit = 0, n_rect = 0, n_hit = 0;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            int64_t b, e;
            LS.span(x, y, b, e);
            T Tr = 1, C[3] = {0, 0, 0}, D = 0, Nv[3] = {0, 0, 0}, Nt[3] = {0, 0, 0}, a_top = 0;
            uint32_t last = 0;
            bool amb = false;
            uint64_t sg = 1469598103934665603ull;
            for (int64_t i = b; i < e; ++i) {
                const Face<T>& f = F[list[i]];
                ++n_visit;
                if (x < f.x0 || x > f.x1 || y < f.y0 || y > f.y1) continue;   // rect is part of the hit rule (S5)
                ++n_rect;
                Hit<T> h;
                if (!eval(f, (T)x, (T)y, face_sigma<T>(prm, list[i]), amin, atol, h, &amb)) continue;
                ++n_hit;
                T wgt = Tr * h.alpha;                                          // Eq. 4
                for (int c = 0; c < 3; ++c) C[c] += wgt * h.c[c];
                D += wgt * h.z;                                                // S11
                if (nrm) for (int c = 0; c < 3; ++c) Nv[c] += wgt * nrm[3 * (int64_t)list[i] + c];   // S26
                if (nrm && h.alpha > a_top) {                                  // S29: the first hit of the largest alpha
                    a_top = h.alpha;
                    for (int c = 0; c < 3; ++c) Nt[c] = nrm[3 * (int64_t)list[i] + c];
                }
                Tr = Tr * ((T)1 - h.alpha);
                last = (uint32_t)(i - b + 1);
                sg = (sg ^ (uint64_t)(list[i] + 1)) * 1099511628211ull;
                if (atol > 0 && tmin > 0 && std::fabs(Tr - tmin) <= atol * tmin) amb = true;
                if (Tr <= tmin) break;                                         // S12: include, then test
            }
            int64_t p = (int64_t)y * W + x;
            if (oc) for (int c = 0; c < 3; ++c) oc[(int64_t)c * W * H + p] = C[c];
            if (od) od[p] = D;
            if (oa) oa[p] = (T)1 - Tr;
            if (on) for (int c = 0; c < 3; ++c) on[(int64_t)c * W * H + p] = Nv[c];
            if (on_top) for (int c = 0; c < 3; ++c) on_top[(int64_t)c * W * H + p] = Nt[c];
            if (n_contrib) n_contrib[p] = last;
            if (ambig) ambig[p] = amb ? 1 : 0;
            if (sig) sig[p] = sg;
        }
    if (counters) counters[0] = n_visit, counters[1] = n_rect, counters[2] = n_hit, counters[3] = 0;
}

// ---------------------------------------------------------------------------------- D-SSIM (Eq. 8)
// L_DSSIM(I, Ibar) = 1 - mean over channels and pixels of SSIM (Eq. 8; the paper only names the
// term, reading S25 of DESIGN.md fixes it as in 3D Gaussian Splatting: 11x11 Gaussian window, sigma 1.5, zero
// padding, C1 = 0.01^2, C2 = 0.03^2, per channel).  Written as the definition: window sums by direct double loops,
// gradient by plain reverse mode of those loops (for every pixel p and every tap q of its window).
// x = rendered image [3][H][W], y = reference.  Returns L; g (may be NULL) receives dL/dx.
template <class T>
double dssim(int32_t W, int32_t H, const T* x, const T* y, T* g) {
    const int R = 5;
    double w1[11], wsum = 0;
    for (int i = 0; i < 11; ++i) wsum += (w1[i] = std::exp(-(double)((i - R) * (i - R)) / (2.0 * 1.5 * 1.5)));
    for (int i = 0; i < 11; ++i) w1[i] /= wsum;
    const T C1 = (T)(0.01 * 0.01), C2 = (T)(0.03 * 0.03);
    const int64_t HW = (int64_t)W * H;
    const double N = 3.0 * (double)HW;
    if (g) for (int64_t i = 0; i < 3 * HW; ++i) g[i] = 0;
    double total = 0;
    for (int c = 0; c < 3; ++c) {
        const T* xc = x + c * HW;
        const T* yc = y + c * HW;
        T* gc = g ? g + c * HW : nullptr;
        for (int py = 0; py < H; ++py)
            for (int px = 0; px < W; ++px) {
                T mu1 = 0, mu2 = 0, e11 = 0, e22 = 0, e12 = 0;
                for (int dy = -R; dy <= R; ++dy)
                    for (int dx = -R; dx <= R; ++dx) {
                        const int qx = px + dx, qy = py + dy;
                        if (qx < 0 || qx >= W || qy < 0 || qy >= H) continue;          // zero padding
                        const T wgt = (T)(w1[dy + R] * w1[dx + R]);
                        const T a = xc[(int64_t)qy * W + qx], b = yc[(int64_t)qy * W + qx];
                        mu1 += wgt * a, mu2 += wgt * b, e11 += wgt * a * a, e22 += wgt * b * b, e12 += wgt * a * b;
                    }
                const T s11 = e11 - mu1 * mu1, s22 = e22 - mu2 * mu2, s12 = e12 - mu1 * mu2;
                const T A1 = 2 * mu1 * mu2 + C1, A2 = 2 * s12 + C2, B1 = mu1 * mu1 + mu2 * mu2 + C1, B2 = s11 + s22 + C2;
                const T ssim = (A1 * A2) / (B1 * B2);
                total += (double)ssim;
                if (!gc) continue;
                // reverse mode: dL/dssim = -1/N; ssim depends on x through mu1, e11 (in s11) and e12 (in s12)
                const T gs = (T)(-1.0 / N);
                const T d_mu1_direct = (2 * mu2 * A2) / (B1 * B2) - (A1 * A2 * 2 * mu1) / (B1 * B1 * B2);
                const T d_s11 = -(A1 * A2) / (B1 * B2 * B2);
                const T d_s12 = (2 * A1) / (B1 * B2);
                // s11 = e11 - mu1^2, s12 = e12 - mu1 mu2
                const T d_mu1 = d_mu1_direct - 2 * mu1 * d_s11 - mu2 * d_s12;
                for (int dy = -R; dy <= R; ++dy)
                    for (int dx = -R; dx <= R; ++dx) {
                        const int qx = px + dx, qy = py + dy;
                        if (qx < 0 || qx >= W || qy < 0 || qy >= H) continue;
                        const T wgt = (T)(w1[dy + R] * w1[dx + R]);
                        const int64_t q = (int64_t)qy * W + qx;
                        gc[q] += gs * wgt * (d_mu1 + d_s11 * 2 * xc[q] + d_s12 * yc[q]);
                    }
            }
    }
    return 1.0 - total / N;
}

// ---------------------------------------------------------------------------------- E_equi (Eq. 14)
// E_equi = 1/|F| sum_m 1/3 sum_n (cos theta_{m,n} - 0.5)^2, cos of the internal angle at vertex n = dot product of the
// normalised edge vectors leaving it, in world space.  Faces with an edge shorter than 1e-12 are
// skipped (no angle).  Returns E; grad_pos[V][3] (may be NULL) += weight * dE/dpos.
template <class T>
double equi(const T* pos, const int32_t* faces, int32_t M, double weight, T* grad_pos) {
    double total = 0;
    for (int m = 0; m < M; ++m) {
        int64_t id[3];
        for (int k = 0; k < 3; ++k) id[k] = vid(faces, m, k);
        T P[3][3];
        for (int k = 0; k < 3; ++k)
            for (int a = 0; a < 3; ++a) P[k][a] = pos[3 * id[k] + a];
        bool ok = true;
        for (int k = 0; k < 3 && ok; ++k) {
            T l2 = 0;
            for (int a = 0; a < 3; ++a) l2 += (P[(k + 1) % 3][a] - P[k][a]) * (P[(k + 1) % 3][a] - P[k][a]);
            ok = l2 > (T)1e-24;
        }
        if (!ok) continue;
        for (int n = 0; n < 3; ++n) {
            const int b = (n + 1) % 3, c = (n + 2) % 3;
            T u[3], v[3], uu = 0, vv = 0, uv = 0;
            for (int a = 0; a < 3; ++a) {
                u[a] = P[b][a] - P[n][a], v[a] = P[c][a] - P[n][a];
                uu += u[a] * u[a], vv += v[a] * v[a], uv += u[a] * v[a];
            }
            const T lu = std::sqrt(uu), lv = std::sqrt(vv), cs = uv / (lu * lv);
            total += (double)((cs - (T)0.5) * (cs - (T)0.5));
            if (!grad_pos) continue;
            const T gcs = (T)(weight / (3.0 * (double)M)) * 2 * (cs - (T)0.5);     // dE/dcos
            for (int a = 0; a < 3; ++a) {
                const T du = v[a] / (lu * lv) - cs * u[a] / uu, dv = u[a] / (lu * lv) - cs * v[a] / vv;
                grad_pos[3 * id[b] + a] += gcs * du;
                grad_pos[3 * id[c] + a] += gcs * dv;
                grad_pos[3 * id[n] + a] -= gcs * (du + dv);
            }
        }
    }
    return total / (3.0 * (double)M);
}

// ---------------------------------------------------------------------------------- per-face statistics
// What the map-management layer of the paper reads off a render (not part of Eq. 1-4): for every face the number of
// pixels it contributed to (the "rendered" flag of the covisibility IoU; the pixel coverage of the
// blur-split test) and its projected area in px^2 (prune test area > eps_a).
// Same walk as render_fwd (same hit rule, same termination); area = |S| / 2 with S of F4.
template <class T>
void face_stats(const T* color, const T* opacity, const int32_t* faces, int32_t M, const tso_camera* cam_,
                const tso_params* prm, const uint8_t* visible, const int16_t* rect, const T* scr, const uint32_t* list,
                int64_t n_list, const uint32_t* tile_ranges, uint32_t* face_pixels, T* proj_area) {
    const Cam<T> cam(cam_);
    const int W = cam.W, H = cam.H;
    const T sigma = (T)prm->sigma, amin = (T)prm->alpha_min, tmin = (T)prm->t_min;
    std::vector<Face<T>> F = setup_all(color, opacity, faces, M, visible, rect, scr, prm->min_opacity != 0);
    Lists<T> LS{list, n_list, tile_ranges, (W + 15) / 16};
    for (int m = 0; m < M; ++m) {
        if (face_pixels) face_pixels[m] = 0;
        if (proj_area) {
            proj_area[m] = 0;
            if (visible[m]) {
                const T* q = scr + 9 * (int64_t)m;                   // (u,v,w) x 3
                const T a = q[3] - q[0], b = q[7] - q[1], c = q[4] - q[1], d = q[6] - q[0];
                const T S = std::fma(a, b, -(c * d));                // F4 / N3
                proj_area[m] = (T)0.5 * std::fabs(S);
            }
        }
    }
    if (!face_pixels) return;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            int64_t b, e;
            LS.span(x, y, b, e);
            T Tr = 1;
            for (int64_t i = b; i < e; ++i) {
                const Face<T>& f = F[list[i]];
                if (x < f.x0 || x > f.x1 || y < f.y0 || y > f.y1) continue;
                Hit<T> h;
                if (!eval(f, (T)x, (T)y, face_sigma<T>(prm, list[i]), amin, (T)0, h, nullptr)) continue;
                face_pixels[list[i]] += 1;
                Tr = Tr * ((T)1 - h.alpha);
                if (Tr <= tmin) break;
            }
        }
}

// ---------------------------------------------------------------------------------- B1..B6
template <class T>
void render_bwd(const T* color, const T* opacity, const int32_t* faces, int32_t M, const tso_camera* cam_,
                const tso_params* prm, const uint8_t* visible, const int16_t* rect, const T* scr,
                const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges, const T* gCi, const T* gDi,
                const T* gAi, T* grad_color, T* grad_opacity, T* g_scr, const T* nrm = nullptr, const T* gNi = nullptr,
                T* g_nrm = nullptr) {
    const Cam<T> cam(cam_);
    const int W = cam.W, H = cam.H;
    const T sigma = (T)prm->sigma, amin = (T)prm->alpha_min, tmin = (T)prm->t_min;
    std::vector<Face<T>> F = setup_all(color, opacity, faces, M, visible, rect, scr, prm->min_opacity != 0);
    Lists<T> LS{list, n_list, tile_ranges, (W + 15) / 16};
    struct Rec { uint32_t m; T Tn; };
    std::vector<Rec> hits;
    for (int y = 0; y < H; ++y)
        for (int x = 0; x < W; ++x) {
            int64_t p = (int64_t)y * W + x;
            T gC[3] = {0, 0, 0}, gD = 0, gA = 0, gN[3] = {0, 0, 0};
            if (nrm && gNi) for (int c = 0; c < 3; ++c) gN[c] = gNi[(int64_t)c * W * H + p];
            if (gCi) for (int c = 0; c < 3; ++c) gC[c] = gCi[(int64_t)c * W * H + p];
            if (gDi) gD = gDi[p];
            if (gAi) gA = gAi[p];
            // forward walk, remembering the transmittance in front of every contributing face
            int64_t b, e;
            LS.span(x, y, b, e);
            hits.clear();
            T Tr = 1;
            Hit<T> h;
            for (int64_t i = b; i < e; ++i) {
                const Face<T>& f = F[list[i]];
                if (x < f.x0 || x > f.x1 || y < f.y0 || y > f.y1) continue;
                if (!eval(f, (T)x, (T)y, face_sigma<T>(prm, list[i]), amin, (T)0, h, nullptr)) continue;
                hits.push_back({list[i], Tr});
                Tr = Tr * ((T)1 - h.alpha);
                if (Tr <= tmin) break;
            }
            // reverse walk; R* = what is composited BEHIND the current face with unit transmittance
            T Rc[3] = {0, 0, 0}, Rd = 0, Ra = 0, Rn[3] = {0, 0, 0};
            for (int64_t j = (int64_t)hits.size() - 1; j >= 0; --j) {
                const uint32_t m = hits[j].m;
                const Face<T>& f = F[m];
                const T Tn = hits[j].Tn;
                const T sigma_m = face_sigma<T>(prm, m);
                eval(f, (T)x, (T)y, sigma_m, amin, (T)0, h, nullptr);
                const T wgt = Tn * h.alpha;
                // B1: vertex colours
                if (grad_color)
                    for (int k = 0; k < 3; ++k)
                        for (int c = 0; c < 3; ++c)
                            grad_color[3 * (int64_t)vid(faces, m, k) + c] += h.lam[k] * wgt * gC[c];
                // B2: dL/dalpha_n
                T ga = 0;
                for (int c = 0; c < 3; ++c) ga += (h.c[c] - Rc[c]) * gC[c];
                ga += (h.z - Rd) * gD + ((T)1 - Ra) * gA;
                if (nrm) {
                    // S26: the face normal is a flat attribute composited like a colour
                    const T* nm = nrm + 3 * (int64_t)m;
                    for (int c = 0; c < 3; ++c) ga += (nm[c] - Rn[c]) * gN[c];
                    for (int c = 0; c < 3; ++c) Rn[c] = h.alpha * nm[c] + ((T)1 - h.alpha) * Rn[c];
                    if (g_nrm) for (int c = 0; c < 3; ++c) g_nrm[3 * (int64_t)m + c] += wgt * gN[c];
                }
                ga *= Tn;
                // B3: push this face onto the "behind" accumulators
                for (int c = 0; c < 3; ++c) Rc[c] = h.alpha * h.c[c] + ((T)1 - h.alpha) * Rc[c];
                Rd = h.alpha * h.z + ((T)1 - h.alpha) * Rd;
                Ra = h.alpha + ((T)1 - h.alpha) * Ra;
                // B4: opacity (mean -> 1/3 each, :82) and window
                if (grad_opacity) {
                    if (f.kmin >= 0) grad_opacity[vid(faces, m, f.kmin)] += h.I * ga;
                    else
                        for (int k = 0; k < 3; ++k) grad_opacity[vid(faces, m, k)] += (h.I / (T)3) * ga;
                }
                const T gI = f.obar * ga;
                const T gx = gI * sigma_m * h.I / h.x;
                // S32: I = x^sigma, so dL/dsigma_m += dL/dI * I ln x
                if (prm->grad_face_sigma) ((T*)prm->grad_face_sigma)[m] += gI * h.I * std::log(h.x);
                // B5: interpolation
                T gom[3], gb[3], gw[3];
                for (int k = 0; k < 3; ++k) {
                    T d = 0;
                    for (int c = 0; c < 3; ++c) d += (f.col[k][c] - h.c[c]) * gC[c];
                    gom[k] = (wgt / h.Om) * (d - h.z * gD);
                    gb[k] = f.w[k] * gom[k];
                    gw[k] = h.b[k] * gom[k];
                }
                // B6: screen-space vertex gradients
                T gqx[3] = {0, 0, 0}, gqy[3] = {0, 0, 0};
                // (i) barycentric path: db_k/dq_j = -b_j grad_p b_k, grad_p b_k = -n_k/h_k
                T Gx = 0, Gy = 0;
                for (int k = 0; k < 3; ++k) Gx += gb[k] * (-f.nx[k] / f.h[k]), Gy += gb[k] * (-f.ny[k] / f.h[k]);
                for (int j2 = 0; j2 < 3; ++j2) gqx[j2] += -h.b[j2] * Gx, gqy[j2] += -h.b[j2] * Gy;
                // (ii) window numerator x = -L_{k*}/r
                {
                    const int ks = h.kstar, a = (ks + 1) % 3, bb = (ks + 2) % 3;
                    const T gL = -gx / f.r;
                    const T ex = f.qx[bb] - f.qx[a], ey = f.qy[bb] - f.qy[a];
                    const T t = (((T)x - f.qx[a]) * ex + ((T)y - f.qy[a]) * ey) / (f.ell[ks] * f.ell[ks]);
                    gqx[a] += -((T)1 - t) * f.nx[ks] * gL, gqy[a] += -((T)1 - t) * f.ny[ks] * gL;
                    gqx[bb] += -t * f.nx[ks] * gL, gqy[bb] += -t * f.ny[ks] * gL;
                }
                // (iii) window denominator r = |S| / sum(ell)
                {
                    const T gr = -(h.x / f.r) * gx;
                    for (int j2 = 0; j2 < 3; ++j2) {
                        const int i1 = (j2 + 1) % 3, i2 = (j2 + 2) % 3;
                        // |q_j - q_{j+1}| is edge (j+2); |q_j - q_{j+2}| is edge (j+1)
                        const T u1x = (f.qx[j2] - f.qx[i1]) / f.ell[i2], u1y = (f.qy[j2] - f.qy[i1]) / f.ell[i2];
                        const T u2x = (f.qx[j2] - f.qx[i2]) / f.ell[i1], u2y = (f.qy[j2] - f.qy[i2]) / f.ell[i1];
                        const T drx = (-f.ell[j2] * f.nx[j2]) / f.sumell - (f.absS / (f.sumell * f.sumell)) * (u1x + u2x);
                        const T dry = (-f.ell[j2] * f.ny[j2]) / f.sumell - (f.absS / (f.sumell * f.sumell)) * (u1y + u2y);
                        gqx[j2] += gr * drx, gqy[j2] += gr * dry;
                    }
                }
                T* gs = g_scr + 9 * (int64_t)m;
                for (int k = 0; k < 3; ++k) gs[3 * k] += gqx[k], gs[3 * k + 1] += gqy[k], gs[3 * k + 2] += gw[k];
            }
        }
}

// ---------------------------------------------------------------------------------- B7..B9
template <class T>
void project_bwd(const int32_t* faces, int32_t M, const T* Tcw, const tso_camera* cam_, const uint8_t* visible,
                 const T* Q, const T* g_scr, T* grad_pos, T* dL_dtau) {
    const Cam<T> cam(cam_);
    T tau[6] = {0, 0, 0, 0, 0, 0};
    for (int m = 0; m < M; ++m) {
        if (!visible[m]) continue;
        for (int k = 0; k < 3; ++k) {
            const T X = Q[9 * (int64_t)m + 3 * k], Y = Q[9 * (int64_t)m + 3 * k + 1], Z = Q[9 * (int64_t)m + 3 * k + 2];
            const T gu = g_scr[9 * (int64_t)m + 3 * k], gv = g_scr[9 * (int64_t)m + 3 * k + 1],
                    gw = g_scr[9 * (int64_t)m + 3 * k + 2];
            // B7: d(u,v,w)/d(X,Y,Z) of Eq. 1 -- the dv_I/dv_C factor of Eq. 5
            const T g[3] = {cam.fx / Z * gu, cam.fy / Z * gv,
                            -cam.fx * X / (Z * Z) * gu - cam.fy * Y / (Z * Z) * gv - gw / (Z * Z)};
            // B8: world, dQ/dP = R
            if (grad_pos) {
                T* gp = grad_pos + 3 * (int64_t)vid(faces, m, k);
                for (int a = 0; a < 3; ++a) gp[a] += Tcw[a] * g[0] + Tcw[4 + a] * g[1] + Tcw[8 + a] * g[2];
            }
            // B9: Eq. 7, Dv_C/DT = [I3, -[v_C]x]  ->  dL/dtau = [g ; Q x g]
            tau[0] += g[0], tau[1] += g[1], tau[2] += g[2];
            tau[3] += Y * g[2] - Z * g[1];
            tau[4] += Z * g[0] - X * g[2];
            tau[5] += X * g[1] - Y * g[0];
        }
    }
    if (dL_dtau) for (int i = 0; i < 6; ++i) dL_dtau[i] = tau[i];
}

// ---------------------------------------------------------------------------------- face normals (Eq. 12)
// The rendered normal map N(V, T_CW) "returned by the rasteriser" (Eq. 12) composites one normal
// per face.  Reading S26 of DESIGN.md: n_m = unit normal of the face plane in CAMERA space, oriented towards the
// camera (n . Q_0 < 0; the plane offset n . Q is the same for every point of the plane).  The edge vectors are taken
// in world space and rotated (R (P_k - P_0) = Q_k - Q_0 exactly, without the cancellation of subtracting two camera-
// space points).  nrm[M][3]; zero for culled faces.
template <class T>
void face_normal(const T* pos, const int32_t* faces, int32_t M, const T* Tcw, const uint8_t* visible, const T* Q,
                 T* nrm) {
    for (int m = 0; m < M; ++m) {
        T* n = nrm + 3 * (int64_t)m;
        n[0] = n[1] = n[2] = 0;
        if (!visible[m]) continue;
        const T* P0 = pos + 3 * (int64_t)vid(faces, m, 0);
        const T* P1 = pos + 3 * (int64_t)vid(faces, m, 1);
        const T* P2 = pos + 3 * (int64_t)vid(faces, m, 2);
        T a[3], b[3];
        for (int i = 0; i < 3; ++i) {
            a[i] = 0, b[i] = 0;
            for (int j = 0; j < 3; ++j) a[i] += Tcw[4 * i + j] * (P1[j] - P0[j]), b[i] += Tcw[4 * i + j] * (P2[j] - P0[j]);
        }
        const T mm[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
        const T len = std::sqrt(mm[0] * mm[0] + mm[1] * mm[1] + mm[2] * mm[2]);
        const T* Q0 = Q + 9 * (int64_t)m;
        const T off = mm[0] * Q0[0] + mm[1] * Q0[1] + mm[2] * Q0[2];
        const T s = off < 0 ? (T)1 : (T)-1;                  // towards the camera
        for (int i = 0; i < 3; ++i) n[i] = s * mm[i] / len;
    }
}

// Reverse mode of face_normal: n = s m/|m|, m = a x b, a = R (P1 - P0), b = R (P2 - P0).
//   g_m = s (g_n - n (n . g_n)) / |m|,  g_a = b x g_m,  g_b = g_m x a   (camera space)
//   grad_pos: P1 += R^T g_a, P2 += R^T g_b, P0 -= R^T (g_a + g_b)
//   pose (left perturbation, Eq. 5-7): a -> Exp(theta) a, so dL/dtheta += a x g_a + b x g_b; no translation term.
// grad_pos (may be NULL) and dL_dtau[6] (may be NULL) are ACCUMULATED into.
template <class T>
void face_normal_bwd(const T* pos, const int32_t* faces, int32_t M, const T* Tcw, const uint8_t* visible, const T* Q,
                     const T* g_nrm, T* grad_pos, T* dL_dtau) {
    for (int m = 0; m < M; ++m) {
        if (!visible[m]) continue;
        const int64_t id0 = vid(faces, m, 0), id1 = vid(faces, m, 1), id2 = vid(faces, m, 2);
        const T *P0 = pos + 3 * id0, *P1 = pos + 3 * id1, *P2 = pos + 3 * id2;
        T a[3], b[3];
        for (int i = 0; i < 3; ++i) {
            a[i] = 0, b[i] = 0;
            for (int j = 0; j < 3; ++j) a[i] += Tcw[4 * i + j] * (P1[j] - P0[j]), b[i] += Tcw[4 * i + j] * (P2[j] - P0[j]);
        }
        const T mm[3] = {a[1] * b[2] - a[2] * b[1], a[2] * b[0] - a[0] * b[2], a[0] * b[1] - a[1] * b[0]};
        const T len = std::sqrt(mm[0] * mm[0] + mm[1] * mm[1] + mm[2] * mm[2]);
        const T* Q0 = Q + 9 * (int64_t)m;
        const T s = (mm[0] * Q0[0] + mm[1] * Q0[1] + mm[2] * Q0[2]) < 0 ? (T)1 : (T)-1;
        T n[3];
        for (int i = 0; i < 3; ++i) n[i] = s * mm[i] / len;
        const T* gn = g_nrm + 3 * (int64_t)m;
        const T ngn = n[0] * gn[0] + n[1] * gn[1] + n[2] * gn[2];
        T gm[3];
        for (int i = 0; i < 3; ++i) gm[i] = s * (gn[i] - n[i] * ngn) / len;
        const T ga[3] = {b[1] * gm[2] - b[2] * gm[1], b[2] * gm[0] - b[0] * gm[2], b[0] * gm[1] - b[1] * gm[0]};
        const T gb[3] = {gm[1] * a[2] - gm[2] * a[1], gm[2] * a[0] - gm[0] * a[2], gm[0] * a[1] - gm[1] * a[0]};
        if (grad_pos) {
            for (int j = 0; j < 3; ++j) {
                const T wa = Tcw[j] * ga[0] + Tcw[4 + j] * ga[1] + Tcw[8 + j] * ga[2];
                const T wb = Tcw[j] * gb[0] + Tcw[4 + j] * gb[1] + Tcw[8 + j] * gb[2];
                grad_pos[3 * id1 + j] += wa, grad_pos[3 * id2 + j] += wb, grad_pos[3 * id0 + j] -= wa + wb;
            }
        }
        if (dL_dtau) {
            dL_dtau[3] += (a[1] * ga[2] - a[2] * ga[1]) + (b[1] * gb[2] - b[2] * gb[1]);
            dL_dtau[4] += (a[2] * ga[0] - a[0] * ga[2]) + (b[2] * gb[0] - b[0] * gb[2]);
            dL_dtau[5] += (a[0] * ga[1] - a[1] * ga[0]) + (b[0] * gb[1] - b[1] * gb[0]);
        }
    }
}

template <class T>
double l1_loss(int32_t W, int32_t H, const T* C, const T* D, const T* Ch, const T* Dh, double lambda_dep, T* gC,
               T* gD) {
    const int64_t n = (int64_t)W * H;
    const T wc = (T)(1.0 / (3.0 * (double)n)), wd = (T)(lambda_dep / (double)n);
    double L = 0;
    for (int64_t i = 0; i < 3 * n; ++i) {
        T d = C[i] - Ch[i];
        L += (double)wc * std::fabs((double)d);
        gC[i] = d > 0 ? wc : (d < 0 ? -wc : (T)0);
    }
    for (int64_t i = 0; i < n; ++i) {
        if (!(Dh[i] > 0)) { gD[i] = 0; continue; }
        T d = D[i] - Dh[i];
        L += (double)wd * std::fabs((double)d);
        gD[i] = d > 0 ? wd : (d < 0 ? -wd : (T)0);
    }
    return L;
}

// E_norm of Eq. 12: sum over the valid pixels of 1 - N_p . Nbar_p.  Reading S27 of DESIGN.md: a pixel
// is valid where the sensor normal exists (Nbar_p != 0), and the sum is divided by H W like the other image terms.
// N, Nbar, gN are [3][H][W]; gN receives weight * dE/dN; returns weight * E_norm.
template <class T>
double normal_loss(int32_t W, int32_t H, const T* N, const T* Nb, double weight, T* gN) {
    const int64_t n = (int64_t)W * H;
    const T w = (T)(weight / (double)n);
    double L = 0;
    for (int64_t i = 0; i < n; ++i) {
        const T b0 = Nb[i], b1 = Nb[n + i], b2 = Nb[2 * n + i];
        const bool valid = b0 != 0 || b1 != 0 || b2 != 0;
        if (valid) L += (double)w * (1.0 - ((double)N[i] * b0 + (double)N[n + i] * b1 + (double)N[2 * n + i] * b2));
        gN[i] = valid ? -w * b0 : (T)0, gN[n + i] = valid ? -w * b1 : (T)0, gN[2 * n + i] = valid ? -w * b2 : (T)0;
    }
    return L;
}

// Screen-space gradient statistic of the densification test (Table S4: "gradient threshold 0.001", "gradient percentile
// 0.99"; the text does not define it).  Reading S28 of DESIGN.md: per face, the norm of the gradient
// of L with respect to a rigid translation of the face in the image plane, ||sum_k (dL/du_k, dL/dv_k)||_2 -- the
// triangle analogue of the view-space point gradient that Gaussian-splatting densification accumulates.
// g_scr[M][9] as written by render_bwd; face_grad2d[M] += the norm, face_views[M] += 1 where the face has a gradient.
template <class T>
void screen_grad_stat(int32_t M, const uint8_t* visible, const T* g_scr, T* face_grad2d, uint32_t* face_views) {
    for (int m = 0; m < M; ++m) {
        if (!visible[m]) continue;
        const T* g = g_scr + 9 * (int64_t)m;
        bool any = false;
        for (int j = 0; j < 9; ++j) any = any || g[j] != 0;
        if (!any) continue;
        const T sx = (g[0] + g[3]) + g[6], sy = (g[1] + g[4]) + g[7];
        face_grad2d[m] += std::sqrt(sx * sx + sy * sy);
        if (face_views) face_views[m] += 1;
    }
}

// SE(3) exponential, tau = (rho, theta).  out = Exp(tau) o T.
template <class T>
void left_perturb(const T* Tcw, const T* tau, T* out) {
    const T rx = tau[0], ry = tau[1], rz = tau[2], wx = tau[3], wy = tau[4], wz = tau[5];
    const T th2 = wx * wx + wy * wy + wz * wz, th = std::sqrt(th2);
    T A, B, Cc;   // sin/th, (1-cos)/th^2, (th-sin)/th^3
    if (th < (T)1e-4) {
        A = (T)1 - th2 / (T)6, B = (T)0.5 - th2 / (T)24, Cc = (T)1 / (T)6 - th2 / (T)120;
    } else {
        A = std::sin(th) / th, B = ((T)1 - std::cos(th)) / th2, Cc = (th - std::sin(th)) / (th2 * th);
    }
    const T K[9] = {0, -wz, wy, wz, 0, -wx, -wy, wx, 0};
    T K2[9];
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) K2[3 * i + j] = K[3 * i] * K[j] + K[3 * i + 1] * K[3 + j] + K[3 * i + 2] * K[6 + j];
    T R[9], Vm[9];
    for (int i = 0; i < 9; ++i) {
        T I = (i % 4 == 0) ? (T)1 : (T)0;
        R[i] = I + A * K[i] + B * K2[i];
        Vm[i] = I + B * K[i] + Cc * K2[i];
    }
    const T tt[3] = {Vm[0] * rx + Vm[1] * ry + Vm[2] * rz, Vm[3] * rx + Vm[4] * ry + Vm[5] * rz,
                     Vm[6] * rx + Vm[7] * ry + Vm[8] * rz};
    for (int i = 0; i < 3; ++i) {
        for (int j = 0; j < 4; ++j) {
            T acc = R[3 * i] * Tcw[j] + R[3 * i + 1] * Tcw[4 + j] + R[3 * i + 2] * Tcw[8 + j];
            out[4 * i + j] = acc + (j == 3 ? tt[i] : (T)0);
        }
    }
}

}  // namespace

// ====================================================================================== C ABI
// Normalised depth (E_dep of Eq. 9 / 13 compares a rendered depth with the sensor depth, and
// D = sum z alpha T under-reads wherever A < 1): Dn = D / A where A > eps, else 0.  Backward of a cotangent gDn:
// gD += gDn / A,  gA += -gDn D / A^2  (nothing where A <= eps).
template <class T>
void depth_normalise(int64_t n, const T* D, const T* A, T eps, T* Dn) {
    for (int64_t i = 0; i < n; ++i) Dn[i] = A[i] > eps ? D[i] / A[i] : (T)0;
}
template <class T>
void depth_normalise_bwd(int64_t n, const T* D, const T* A, T eps, const T* gDn, T* gD, T* gA) {
    for (int64_t i = 0; i < n; ++i) {
        if (!(A[i] > eps)) continue;
        gD[i] += gDn[i] / A[i];
        gA[i] += -gDn[i] * D[i] / (A[i] * A[i]);
    }
}

template <class T>
int64_t bin_sort_impl(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect, const uint32_t* depth_key,
                      const T* scr, int tight, uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
    const int tiles_x = (W + 15) / 16, tiles_y = (H + 15) / 16, NT = tiles_x * tiles_y;
    struct KV { uint64_t k; uint32_t v; };
    std::vector<KV> pairs;
    for (int m = 0; m < M; ++m) {
        if (!visible[m]) continue;
        const int16_t* rc = rect + 4 * (int64_t)m;
        T u[3] = {0, 0, 0}, v[3] = {0, 0, 0};
        if (tight)
            for (int k = 0; k < 3; ++k) u[k] = scr[9 * (int64_t)m + 3 * k], v[k] = scr[9 * (int64_t)m + 3 * k + 1];
        for (int ty = rc[1] >> 4; ty <= (rc[3] >> 4); ++ty)
            for (int tx = rc[0] >> 4; tx <= (rc[2] >> 4); ++tx)
                if (tile_included<T>(tight != 0, u, v, rc, tx, ty))
                    pairs.push_back({((uint64_t)(ty * tiles_x + tx) << 32) | depth_key[m], (uint32_t)m});
    }
    std::stable_sort(pairs.begin(), pairs.end(), [](const KV& a, const KV& b) { return a.k < b.k; });
    for (int t = 0; t < 2 * NT; ++t) ranges[t] = 0;
    const int64_t P = (int64_t)pairs.size();
    for (int64_t i = 0; i < P; ++i) {
        keys[i] = pairs[i].k, vals[i] = pairs[i].v;
        uint32_t t = (uint32_t)(pairs[i].k >> 32);
        if (i == 0 || (uint32_t)(pairs[i - 1].k >> 32) != t) ranges[2 * t] = (uint32_t)i;
        ranges[2 * t + 1] = (uint32_t)(i + 1);
    }
    return P;
}

extern "C" {

int64_t tso_project_f32(const float* pos, const int32_t* faces, int32_t, int32_t M, const float* T_cw,
                        const tso_camera* cam, const tso_params* prm, uint8_t* visible, int16_t* rect,
                        uint32_t* depth_key, uint32_t* tiles_touched, float* scr, float* Q, float* zbar) {
    return project<float>(pos, faces, M, T_cw, cam, prm, visible, rect, depth_key, tiles_touched, scr, Q, zbar);
}
int64_t tso_project_f64(const double* pos, const int32_t* faces, int32_t, int32_t M, const double* T_cw,
                        const tso_camera* cam, const tso_params* prm, uint8_t* visible, int16_t* rect,
                        uint32_t* depth_key, uint32_t* tiles_touched, double* scr, double* Q, double* zbar) {
    return project<double>(pos, faces, M, T_cw, cam, prm, visible, rect, depth_key, tiles_touched, scr, Q, zbar);
}

int64_t tso_bin_sort(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect,
                     const uint32_t* depth_key, const uint32_t* tiles_touched, uint64_t* keys, uint32_t* vals,
                     uint32_t* ranges) {
    (void)tiles_touched;
    return bin_sort_impl<float>(M, W, H, visible, rect, depth_key, nullptr, 0, keys, vals, ranges);
}
int64_t tso_bin_sort_tight_f32(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect,
                               const uint32_t* depth_key, const float* scr, uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
    return bin_sort_impl<float>(M, W, H, visible, rect, depth_key, scr, 1, keys, vals, ranges);
}
int64_t tso_bin_sort_tight_f64(int32_t M, int32_t W, int32_t H, const uint8_t* visible, const int16_t* rect,
                               const uint32_t* depth_key, const double* scr, uint64_t* keys, uint32_t* vals, uint32_t* ranges) {
    return bin_sort_impl<double>(M, W, H, visible, rect, depth_key, scr, 1, keys, vals, ranges);
}

#define TSO_FWD_ARGS color, opacity, faces, M, cam, prm, visible, rect, scr, list, n_list, tile_ranges
void tso_render_fwd_f32(const float* color, const float* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const float* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        float* out_color, float* out_depth, float* out_alpha, uint32_t* n_contrib, uint8_t* ambig,
                        uint64_t* sig, uint64_t* counters) {
    render_fwd<float>(TSO_FWD_ARGS, out_color, out_depth, out_alpha, n_contrib, ambig, sig, counters);
}
void tso_render_fwd_f64(const double* color, const double* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const double* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        double* out_color, double* out_depth, double* out_alpha, uint32_t* n_contrib,
                        uint8_t* ambig, uint64_t* sig, uint64_t* counters) {
    render_fwd<double>(TSO_FWD_ARGS, out_color, out_depth, out_alpha, n_contrib, ambig, sig, counters);
}
void tso_render_bwd_f32(const float* color, const float* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const float* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        const float* dL_dcolor, const float* dL_ddepth, const float* dL_dalpha, float* grad_color,
                        float* grad_opacity, float* g_scr) {
    render_bwd<float>(TSO_FWD_ARGS, dL_dcolor, dL_ddepth, dL_dalpha, grad_color, grad_opacity, g_scr);
}
void tso_render_bwd_f64(const double* color, const double* opacity, const int32_t* faces, int32_t M,
                        const tso_camera* cam, const tso_params* prm, const uint8_t* visible, const int16_t* rect,
                        const double* scr, const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges,
                        const double* dL_dcolor, const double* dL_ddepth, const double* dL_dalpha,
                        double* grad_color, double* grad_opacity, double* g_scr) {
    render_bwd<double>(TSO_FWD_ARGS, dL_dcolor, dL_ddepth, dL_dalpha, grad_color, grad_opacity, g_scr);
}

void tso_project_bwd_f32(const int32_t* faces, int32_t M, const float* T_cw, const tso_camera* cam,
                         const uint8_t* visible, const float* Q, const float* g_scr, float* grad_pos,
                         float* dL_dtau) {
    project_bwd<float>(faces, M, T_cw, cam, visible, Q, g_scr, grad_pos, dL_dtau);
}
void tso_project_bwd_f64(const int32_t* faces, int32_t M, const double* T_cw, const tso_camera* cam,
                         const uint8_t* visible, const double* Q, const double* g_scr, double* grad_pos,
                         double* dL_dtau) {
    project_bwd<double>(faces, M, T_cw, cam, visible, Q, g_scr, grad_pos, dL_dtau);
}

double tso_l1_loss_f32(int32_t W, int32_t H, const float* C, const float* D, const float* Chat, const float* Dhat,
                       double lambda_dep, float* gC, float* gD) {
    return l1_loss<float>(W, H, C, D, Chat, Dhat, lambda_dep, gC, gD);
}
double tso_l1_loss_f64(int32_t W, int32_t H, const double* C, const double* D, const double* Chat,
                       const double* Dhat, double lambda_dep, double* gC, double* gD) {
    return l1_loss<double>(W, H, C, D, Chat, Dhat, lambda_dep, gC, gD);
}

void tso_pose_step_f32(float* T_cw, const float* g, float* state, const float* lr, float beta1, float beta2,
                       float eps) {
    float* m = state;
    float* v = state + 6;
    state[12] += 1.0f;
    const float t = state[12];
    const float c1 = 1.0f - std::pow(beta1, t), c2 = 1.0f - std::pow(beta2, t);
    float delta[6];
    for (int i = 0; i < 6; ++i) {
        m[i] = beta1 * m[i] + (1.0f - beta1) * g[i];
        v[i] = beta2 * v[i] + (1.0f - beta2) * g[i] * g[i];
        const float mh = m[i] / c1, vh = v[i] / c2;
        delta[i] = -lr[i] * mh / (std::sqrt(vh) + eps);
    }
    float T4[12];
    left_perturb<float>(T_cw, delta, T4);
    for (int i = 0; i < 12; ++i) T_cw[i] = T4[i];
}

void tso_depth_normalise_f32(int64_t n, const float* D, const float* A, float eps, float* Dn) { depth_normalise<float>(n, D, A, eps, Dn); }
void tso_depth_normalise_f64(int64_t n, const double* D, const double* A, double eps, double* Dn) { depth_normalise<double>(n, D, A, eps, Dn); }
void tso_depth_normalise_bwd_f32(int64_t n, const float* D, const float* A, float eps, const float* gDn, float* gD, float* gA) {
    depth_normalise_bwd<float>(n, D, A, eps, gDn, gD, gA);
}
void tso_depth_normalise_bwd_f64(int64_t n, const double* D, const double* A, double eps, const double* gDn, double* gD, double* gA) {
    depth_normalise_bwd<double>(n, D, A, eps, gDn, gD, gA);
}

void tso_left_perturb_f64(const double* T_cw, const double* tau, double* out) { left_perturb<double>(T_cw, tau, out); }

double tso_equi_f32(const float* pos, const int32_t* faces, int32_t M, double weight, float* grad_pos) {
    return equi<float>(pos, faces, M, weight, grad_pos);
}
double tso_equi_f64(const double* pos, const int32_t* faces, int32_t M, double weight, double* grad_pos) {
    return equi<double>(pos, faces, M, weight, grad_pos);
}

double tso_dssim_f32(int32_t W, int32_t H, const float* x, const float* y, float* g) { return dssim<float>(W, H, x, y, g); }
double tso_dssim_f64(int32_t W, int32_t H, const double* x, const double* y, double* g) { return dssim<double>(W, H, x, y, g); }

void tso_face_stats_f32(const float* color, const float* opacity, const int32_t* faces, int32_t M, const tso_camera* cam,
                        const tso_params* prm, const uint8_t* visible, const int16_t* rect, const float* scr,
                        const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges, uint32_t* face_pixels,
                        float* proj_area) {
    face_stats<float>(color, opacity, faces, M, cam, prm, visible, rect, scr, list, n_list, tile_ranges, face_pixels, proj_area);
}
void tso_face_stats_f64(const double* color, const double* opacity, const int32_t* faces, int32_t M, const tso_camera* cam,
                        const tso_params* prm, const uint8_t* visible, const int16_t* rect, const double* scr,
                        const uint32_t* list, int64_t n_list, const uint32_t* tile_ranges, uint32_t* face_pixels,
                        double* proj_area) {
    face_stats<double>(color, opacity, faces, M, cam, prm, visible, rect, scr, list, n_list, tile_ranges, face_pixels, proj_area);
}

#define TSO_NRM_FWD(T, sfx)                                                                                            \
    void tso_face_normal_##sfx(const T* pos, const int32_t* faces, int32_t M, const T* T_cw, const uint8_t* visible,  \
                               const T* Q, T* nrm) {                                                                   \
        face_normal<T>(pos, faces, M, T_cw, visible, Q, nrm);                                                          \
    }                                                                                                                  \
    void tso_face_normal_bwd_##sfx(const T* pos, const int32_t* faces, int32_t M, const T* T_cw,                       \
                                   const uint8_t* visible, const T* Q, const T* g_nrm, T* grad_pos, T* dL_dtau) {      \
        face_normal_bwd<T>(pos, faces, M, T_cw, visible, Q, g_nrm, grad_pos, dL_dtau);                                 \
    }                                                                                                                  \
    void tso_render_normal_fwd_##sfx(const T* color, const T* opacity, const int32_t* faces, int32_t M,                \
                                     const tso_camera* cam, const tso_params* prm, const uint8_t* visible,             \
                                     const int16_t* rect, const T* scr, const uint32_t* list, int64_t n_list,          \
                                     const uint32_t* tile_ranges, const T* nrm, T* out_normal) {                       \
        render_fwd<T>(TSO_FWD_ARGS, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nrm, out_normal);   \
    }                                                                                                                  \
    void tso_render_normal_top_##sfx(const T* color, const T* opacity, const int32_t* faces, int32_t M,                \
                                     const tso_camera* cam, const tso_params* prm, const uint8_t* visible,             \
                                     const int16_t* rect, const T* scr, const uint32_t* list, int64_t n_list,          \
                                     const uint32_t* tile_ranges, const T* nrm, T* out_normal_top) {                   \
        render_fwd<T>(TSO_FWD_ARGS, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nrm, nullptr,       \
                      out_normal_top);                                                                                 \
    }                                                                                                                  \
    void tso_render_normal_bwd_##sfx(const T* color, const T* opacity, const int32_t* faces, int32_t M,                \
                                     const tso_camera* cam, const tso_params* prm, const uint8_t* visible,             \
                                     const int16_t* rect, const T* scr, const uint32_t* list, int64_t n_list,          \
                                     const uint32_t* tile_ranges, const T* nrm, const T* dL_dnormal, T* grad_opacity,  \
                                     T* g_scr, T* g_nrm) {                                                             \
        render_bwd<T>(TSO_FWD_ARGS, nullptr, nullptr, nullptr, nullptr, grad_opacity, g_scr, nrm, dL_dnormal, g_nrm);  \
    }
TSO_NRM_FWD(float, f32)
TSO_NRM_FWD(double, f64)

void tso_screen_grad_stat_f32(int32_t M, const uint8_t* visible, const float* g_scr, float* face_grad2d, uint32_t* face_views) {
    screen_grad_stat<float>(M, visible, g_scr, face_grad2d, face_views);
}
void tso_screen_grad_stat_f64(int32_t M, const uint8_t* visible, const double* g_scr, double* face_grad2d, uint32_t* face_views) {
    screen_grad_stat<double>(M, visible, g_scr, face_grad2d, face_views);
}

double tso_normal_loss_f32(int32_t W, int32_t H, const float* N, const float* Nbar, double weight, float* gN) {
    return normal_loss<float>(W, H, N, Nbar, weight, gN);
}
double tso_normal_loss_f64(int32_t W, int32_t H, const double* N, const double* Nbar, double weight, double* gN) {
    return normal_loss<double>(W, H, N, Nbar, weight, gN);
}

}  // extern "C"
