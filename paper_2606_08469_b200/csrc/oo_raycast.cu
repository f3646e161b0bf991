// oo_raycast.cu — row f5: primary visibility of the analytic stand-in scene as a CUDA kernel that writes the queries
// (x, n, wo) straight into the caller's device buffers, so a frame never crosses PCIe ("standard primary visibility",
// PAPER.md P:202; the paper itself traces its G-buffers with Mitsuba 3).
//
// One thread per pixel, scanline order.  Double precision with every operation rounded on its own (__dmul_rn /
// __dadd_rn / IEEE division and square root; nothing contracted into an FMA), summed left to right, so the result is
// the one the definition gives on any IEEE machine:
//   d = normalize(f + px r + py u),  px = (2(i+1/2)/W - 1) th aspect,  py = (1 - 2(j+1/2)/H) th
//   sphere: oc = o - c, b = oc.d, cc = oc.oc - R^2, disc = b^2 - cc >= 0, t = -b - sqrt(disc) (or -b + sqrt(disc) if <= tmin)
//   plane : t = (p - o_a)/d_a, accepted if the other two coordinates of o + t d lie in [lo, hi]
//   nearest t > tmin = 1e-9, spheres in order then the planes x=lo, x=hi, y=lo, y=hi, z=lo; strict '<' replaces.
// The sphere list sits in shared memory; oc.oc - R^2 does not depend on the pixel and is precomputed per block.
// Culling: a sphere whose fp32 discriminant is below -64 eps32 (|oc|^2 + R^2) cannot have a non-negative fp64 discriminant
// (the fp32 evaluation is off by at most ~10 eps32 |oc|^2), so it is skipped without touching the fp64 pipe; every
// sphere that passes is decided by the fp64 sequence above, so the result is unchanged.
#include "oo_device.cuh"

namespace oo {

struct RayCam {
    double eye[3], f[3], r[3], u[3];
    double th, aspect, lo, hi;
    uint32_t width, height, n_spheres, pad_;
};

constexpr int kRayThreads = 128;

__device__ __forceinline__ double dot3(double ax, double ay, double az, double bx, double by, double bz) {
    return __dadd_rn(__dadd_rn(__dmul_rn(ax, bx), __dmul_rn(ay, by)), __dmul_rn(az, bz));
}

__global__ void __launch_bounds__(kRayThreads) raycast_kernel(const __grid_constant__ RayCam C, const double* __restrict__ spheres,
                                                              float* __restrict__ x, float* __restrict__ nrm, float* __restrict__ wo,
                                                              int32_t* __restrict__ surf) {
    extern __shared__ __align__(16) double s_sph[];          // [n][8]: cx cy cz R | ocx ocy ocz cc ; then float [n][4]: oc, cc; thr
    float* s_f = (float*)(s_sph + 8 * (size_t)C.n_spheres);   // [n][8] floats: ocx ocy ocz cc thr - - -
    for (uint32_t s = threadIdx.x; s < C.n_spheres; s += kRayThreads) {
        const double cx = spheres[4 * s], cy = spheres[4 * s + 1], cz = spheres[4 * s + 2], R = spheres[4 * s + 3];
        const double ox = __dsub_rn(C.eye[0], cx), oy = __dsub_rn(C.eye[1], cy), oz = __dsub_rn(C.eye[2], cz);
        double* p = s_sph + 8 * s;
        p[0] = cx; p[1] = cy; p[2] = cz; p[3] = R;
        p[4] = ox; p[5] = oy; p[6] = oz;
        p[7] = __dsub_rn(dot3(ox, oy, oz, ox, oy, oz), __dmul_rn(R, R));
        float* pf = s_f + 8 * s;
        pf[0] = (float)ox; pf[1] = (float)oy; pf[2] = (float)oz; pf[3] = (float)p[7];
        pf[4] = -64.0f * 1.1920929e-7f * (float)(dot3(ox, oy, oz, ox, oy, oz) + R * R);
    }
    __syncthreads();
    const uint64_t n = (uint64_t)C.width * C.height;
    const uint64_t q = blockIdx.x * (uint64_t)kRayThreads + threadIdx.x;
    if (q >= n) return;
    const uint32_t j = (uint32_t)(q / C.width), i = (uint32_t)(q - (uint64_t)j * C.width);
    const double px = __dmul_rn(__dmul_rn(__dsub_rn(__ddiv_rn(__dmul_rn(2.0, __dadd_rn((double)i, 0.5)), (double)C.width), 1.0), C.th), C.aspect);
    const double py = __dmul_rn(__dsub_rn(1.0, __ddiv_rn(__dmul_rn(2.0, __dadd_rn((double)j, 0.5)), (double)C.height)), C.th);
    double d[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) d[a] = __dadd_rn(__dadd_rn(C.f[a], __dmul_rn(px, C.r[a])), __dmul_rn(py, C.u[a]));
    {
        const double l = __dsqrt_rn(dot3(d[0], d[1], d[2], d[0], d[1], d[2]));
#pragma unroll
        for (int a = 0; a < 3; ++a) d[a] = __ddiv_rn(d[a], l);
    }
    const double tmin = 1e-9;
    double best = __longlong_as_double(0x7ff0000000000000ll);
    int bs = -1;
    const float df[3] = {(float)d[0], (float)d[1], (float)d[2]};
    for (uint32_t s = 0; s < C.n_spheres; ++s) {
        const float4 cf = *(const float4*)(s_f + 8 * s);
        const float bf = cf.x * df[0] + cf.y * df[1] + cf.z * df[2];
        if (bf * bf - cf.w < s_f[8 * s + 4]) continue;
        const double* p = s_sph + 8 * s;
        const double b = dot3(p[4], p[5], p[6], d[0], d[1], d[2]);
        const double disc = __dsub_rn(__dmul_rn(b, b), p[7]);
        if (disc < 0.0) continue;
        const double sq = __dsqrt_rn(disc);
        double t = __dsub_rn(-b, sq);
        if (t <= tmin) t = __dadd_rn(-b, sq);
        if (t > tmin && t < best) { best = t; bs = (int)s; }
    }
#pragma unroll
    for (int p = 0; p < 5; ++p) {
        const int ax = p >> 1;                               // x, x, y, y, z
        const double pos = (p & 1) ? C.hi : C.lo;            // lo, hi, lo, hi, lo
        if (d[ax] == 0.0) continue;
        const double t = __ddiv_rn(__dsub_rn(pos, C.eye[ax]), d[ax]);
        if (t <= tmin || t >= best) continue;
        bool ok = true;
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            if (a == ax) continue;
            const double v = __dadd_rn(C.eye[a], __dmul_rn(t, d[a]));
            if (v < C.lo || v > C.hi) ok = false;
        }
        if (ok) { best = t; bs = (int)C.n_spheres + p; }
    }
    float ox[3] = {0.0f, 0.0f, 0.0f}, on[3] = {0.0f, 0.0f, 0.0f}, ow[3] = {0.0f, 0.0f, 0.0f};
    if (bs >= 0) {
        double h[3];
#pragma unroll
        for (int a = 0; a < 3; ++a) {
            h[a] = __dadd_rn(C.eye[a], __dmul_rn(best, d[a]));
            ox[a] = __double2float_rn(h[a]);
            ow[a] = __double2float_rn(-d[a]);
        }
        if (bs < (int)C.n_spheres) {
            const double* p = s_sph + 8 * bs;
#pragma unroll
            for (int a = 0; a < 3; ++a) on[a] = __double2float_rn(__ddiv_rn(__dsub_rn(h[a], p[a]), p[3]));
        } else {
            const int p = bs - (int)C.n_spheres;
            const float v = (p & 1) ? -1.0f : 1.0f;
            on[0] = (p >> 1) == 0 ? v : 0.0f;
            on[1] = (p >> 1) == 1 ? v : 0.0f;
            on[2] = (p >> 1) == 2 ? v : 0.0f;
        }
    }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        x[q * 3 + a] = ox[a];
        nrm[q * 3 + a] = on[a];
        wo[q * 3 + a] = ow[a];
    }
    if (surf) surf[q] = bs;
}

// Host side: camera basis in double (f = normalize(look - eye), r = normalize(f x up), u = r x f, th = tan(vfov/2)).
int launch_raycast(const double* d_spheres, uint32_t n_spheres, double lo, double hi, const double eye[3], const double look[3],
                   const double up[3], double vfov_deg, uint32_t width, uint32_t height, float* x, float* nrm, float* wo,
                   int32_t* surf, cudaStream_t stream) {
    const uint64_t n = (uint64_t)width * height;
    if (n == 0) return 0;
    RayCam C{};
    auto norm = [](double v[3]) {
        const double l = sqrt((v[0] * v[0] + v[1] * v[1]) + v[2] * v[2]);
        v[0] /= l; v[1] /= l; v[2] /= l;
    };
    for (int a = 0; a < 3; ++a) { C.eye[a] = eye[a]; C.f[a] = look[a] - eye[a]; }
    norm(C.f);
    C.r[0] = C.f[1] * up[2] - C.f[2] * up[1];
    C.r[1] = C.f[2] * up[0] - C.f[0] * up[2];
    C.r[2] = C.f[0] * up[1] - C.f[1] * up[0];
    norm(C.r);
    C.u[0] = C.r[1] * C.f[2] - C.r[2] * C.f[1];
    C.u[1] = C.r[2] * C.f[0] - C.r[0] * C.f[2];
    C.u[2] = C.r[0] * C.f[1] - C.r[1] * C.f[0];
    C.th = tan(0.5 * vfov_deg * 3.14159265358979323846 / 180.0);
    C.aspect = (double)width / (double)height;
    C.lo = lo; C.hi = hi; C.width = width; C.height = height; C.n_spheres = n_spheres;
    const uint32_t smem = n_spheres * (8 * sizeof(double) + 8 * sizeof(float));
    if (smem > 220 * 1024) return -1;
    static std::atomic<uint64_t> opted{0};
    if (!opt_in_smem(opted, (const void*)raycast_kernel, 220 * 1024)) return kLaunchCudaError;
    raycast_kernel<<<(unsigned)((n + kRayThreads - 1) / kRayThreads), kRayThreads, smem, stream>>>(C, d_spheres, x, nrm, wo, surf);
    return 1;
}

}  // namespace oo
