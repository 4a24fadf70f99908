// Iso-surface ray-caster (Fig. 5: the drops are shown as the iso-surface phi = 0).
// Pure compute: one thread per pixel marches a ray through the physical-space field held in device memory and writes
// intensity and depth into headless device buffers; no graphics API.  The algorithm (camera, slab intersection,
// trilinear sampling on the Fourier x Fourier x Gauss-Lobatto grid, fixed-step march, 24 bisections, central-difference
// normal, 0.2 + 0.8 |n . l| shading) is stated in include/psdns.h; the oracle restates it independently in numpy.
#pragma once
#include <cuda_runtime.h>

namespace psdns {

constexpr int RC_NBIS = 24;

struct RayArgs {
    const double *phi;      // [nz][ny][nx]
    const double *zn;       // z_k = cos(pi k / N), k = 0..N
    double *intensity, *depth;   // [height][width]
    int nx, ny, nz;
    double lx, ly;
    double eye[3], fwd[3], right[3], upv[3], light[3];   // unit vectors, prepared on the host
    double tan_half, aspect, step, iso;
    int width, height;
};

struct V3 { double x, y, z; };
__device__ __forceinline__ V3 v3(double x, double y, double z) { V3 r; r.x = x; r.y = y; r.z = z; return r; }

__device__ __forceinline__ double rc_sample(const RayArgs &a, double px, double py, double pz) {
    const int N = a.nz - 1;
    const double fx = px / (a.lx / a.nx), fy = py / (a.ly / a.ny);
    const double ix = floor(fx), iy = floor(fy);
    const double wx = fx - ix, wy = fy - iy;
    long long i0 = (long long)ix % a.nx; if (i0 < 0) i0 += a.nx;
    long long j0 = (long long)iy % a.ny; if (j0 < 0) j0 += a.ny;
    const int i1 = (int)((i0 + 1) % a.nx), j1 = (int)((j0 + 1) % a.ny);
    const double z = fmin(fmax(pz, -1.0), 1.0);
    int k = (int)floor(acos(z) * ((double)N / 3.14159265358979323846));
    k = min(max(k, 0), N - 1);
#pragma unroll
    for (int r = 0; r < 2; ++r) {              // repair a rounding slip of acos at a node
        if (z > a.zn[k] && k > 0) --k;
        if (z < a.zn[k + 1] && k < N - 1) ++k;
    }
    const double wz = (a.zn[k] - z) / (a.zn[k] - a.zn[k + 1]);
    const size_t pl = (size_t)a.ny * a.nx;
    const double *p0 = a.phi + (size_t)k * pl, *p1 = p0 + pl;
    const size_t r0 = (size_t)j0 * a.nx, r1 = (size_t)j1 * a.nx;
    const double a0 = p0[r0 + i0] * (1.0 - wx) + p0[r0 + i1] * wx, b0 = p0[r1 + i0] * (1.0 - wx) + p0[r1 + i1] * wx;
    const double a1 = p1[r0 + i0] * (1.0 - wx) + p1[r0 + i1] * wx, b1 = p1[r1 + i0] * (1.0 - wx) + p1[r1 + i1] * wx;
    const double lo = a0 * (1.0 - wy) + b0 * wy, hi = a1 * (1.0 - wy) + b1 * wy;
    return lo * (1.0 - wz) + hi * wz;
}

__global__ void __launch_bounds__(128) k_raycast(const __grid_constant__ RayArgs a) {
    const int pix = blockIdx.x * blockDim.x + threadIdx.x;
    if (pix >= a.width * a.height) return;
    const int px = pix % a.width, py = pix / a.width;
    const double sx = (2.0 * (px + 0.5) / a.width - 1.0) * a.tan_half * a.aspect;
    const double sy = (1.0 - 2.0 * (py + 0.5) / a.height) * a.tan_half;
    double d[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) d[c] = a.fwd[c] + sx * a.right[c] + sy * a.upv[c];
    const double dn = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
#pragma unroll
    for (int c = 0; c < 3; ++c) d[c] /= dn;
    // slab intersection with [0, lx] x [0, ly] x [-1, 1]
    const double lo[3] = {0.0, 0.0, -1.0}, hi[3] = {a.lx, a.ly, 1.0};
    double t0 = 0.0, t1 = INFINITY;
    bool alive = true;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        if (d[c] == 0.0) {
            if (a.eye[c] < lo[c] || a.eye[c] > hi[c]) alive = false;
        } else {
            const double inv = 1.0 / d[c];
            const double ta = (lo[c] - a.eye[c]) * inv, tb = (hi[c] - a.eye[c]) * inv;
            t0 = fmax(t0, fmin(ta, tb));
            t1 = fmin(t1, fmax(ta, tb));
        }
    }
    alive = alive && (t1 > t0);
    double inten = 0.0, depth = -1.0;
    if (alive) {
        auto g = [&](double t) { return rc_sample(a, a.eye[0] + t * d[0], a.eye[1] + t * d[1], a.eye[2] + t * d[2]) - a.iso; };
        double tp = t0, gp = g(t0);
        bool found = false;
        double ta = 0.0, tb = 0.0, ga = 0.0;
        for (int i = 1; tp < t1; ++i) {
            const double t = fmin(t0 + i * a.step, t1);
            const double gv = g(t);
            if ((gp < 0.0) != (gv < 0.0)) { found = true; ta = tp; tb = t; ga = gp; break; }
            gp = gv; tp = t;
        }
        if (found) {
            for (int b = 0; b < RC_NBIS; ++b) {
                const double tm = 0.5 * (ta + tb), gm = g(tm);
                if ((gm < 0.0) == (ga < 0.0)) { ta = tm; ga = gm; } else tb = tm;
            }
            const double th = 0.5 * (ta + tb);
            const double p[3] = {a.eye[0] + th * d[0], a.eye[1] + th * d[1], a.eye[2] + th * d[2]};
            const double h[3] = {a.lx / a.nx, a.ly / a.ny, 1.0 / (a.nz - 1)};
            double gr[3];
            gr[0] = (rc_sample(a, p[0] + h[0], p[1], p[2]) - rc_sample(a, p[0] - h[0], p[1], p[2])) / (2.0 * h[0]);
            gr[1] = (rc_sample(a, p[0], p[1] + h[1], p[2]) - rc_sample(a, p[0], p[1] - h[1], p[2])) / (2.0 * h[1]);
            gr[2] = (rc_sample(a, p[0], p[1], p[2] + h[2]) - rc_sample(a, p[0], p[1], p[2] - h[2])) / (2.0 * h[2]);
            const double gn = sqrt(gr[0] * gr[0] + gr[1] * gr[1] + gr[2] * gr[2]);
            inten = gn > 0.0 ? 0.2 + 0.8 * fabs((gr[0] * a.light[0] + gr[1] * a.light[1] + gr[2] * a.light[2]) / gn) : 0.2;
            depth = th;
        }
    }
    a.intensity[pix] = inten;
    a.depth[pix] = depth;
}

}  // namespace psdns
