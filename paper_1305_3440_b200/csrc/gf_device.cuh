// gf_device.cuh -- device-side building blocks of libgf_b200: lattice geometry, the private
// link layout, 3x3 complex algebra in registers, the SU(2) subgroup step and Philox4x32-10.
// Written for sm_100a only.  Citations "PAPER.md:<line>" refer to arXiv:1305.3440.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

namespace gf {

// ------------------------------------------------------------------------------ fast division
// Unsigned division by a run-time constant (Granlund-Montgomery): q = (t + ((n - t) >> s1)) >> s2
// with t = mulhi(n, m).  Exact for every 32-bit n.
struct FastDiv {
    uint32_t d, m, s1, s2;
};

inline FastDiv make_fastdiv(uint32_t d)
{
    FastDiv f;
    f.d = d;
    uint32_t l = 0;
    while ((uint64_t(1) << l) < d) ++l;
    f.m = uint32_t(((uint64_t(1) << 32) * ((uint64_t(1) << l) - d)) / d + 1);
    f.s1 = l < 1 ? l : 1;
    f.s2 = l > 0 ? l - 1 : 0;
    return f;
}

__device__ __forceinline__ uint32_t fdiv(uint32_t n, const FastDiv& f)
{
    const uint32_t t = __umulhi(n, f.m);
    return (t + ((n - t) >> f.s1)) >> f.s2;
}

// ---------------------------------------------------------------------------------- geometry
// Sites of one parity are numbered by the half-index h = s >> 1, s = x + Nx (y + Ny (z + Nz t)),
// so h = xh + nxh (y + Ny (z + Nz t)) with xh = x >> 1, nxh = Nx/2, and
// x = 2 xh + ((y + z + t + parity) & 1).  Time slices are contiguous in h.
struct Geom {
    uint32_t nxh, ny, nz, nt;   // Nx/2, Ny, Nz, Nt
    uint32_t Vh;                // sites per parity
    uint32_t Vp[2];             // Vh rounded up to whole layout tiles: [0] fp32 (64 sites), [1] fp64 (32 sites)
    uint32_t stride[4];         // distance in h of one step in mu (mu=1: unused)
    uint32_t extent[4];         // N_mu
    FastDiv div_nxh, div_ny, div_nz;
    uint32_t sh;                // sites per time slice per parity = Vh / Nt
    FastDiv div_sh;
};

struct Site {
    uint32_t h, xh, c[4];       // c[mu]: c[0]=t, c[1]=x, c[2]=y, c[3]=z
    uint32_t xodd;              // x & 1
};

__device__ __forceinline__ Site decode_site(const Geom& G, uint32_t h, uint32_t parity)
{
    Site s;
    s.h = h;
    const uint32_t r0 = fdiv(h, G.div_nxh);
    s.xh = h - r0 * G.nxh;
    const uint32_t r1 = fdiv(r0, G.div_ny);
    s.c[2] = r0 - r1 * G.ny;
    s.c[0] = fdiv(r1, G.div_nz);
    s.c[3] = r1 - s.c[0] * G.nz;
    s.xodd = (s.c[2] + s.c[3] + s.c[0] + parity) & 1u;
    s.c[1] = 2u * s.xh + s.xodd;
    return s;
}

// c[mu] for a run-time mu without indexing the register array dynamically
__device__ __forceinline__ uint32_t coord(const Site& s, int mu)
{
    return mu == 0 ? s.c[0] : mu == 2 ? s.c[2] : mu == 3 ? s.c[3] : s.c[1];
}

// half-index of x - mu_hat (which has the opposite parity), periodic
__device__ __forceinline__ uint32_t backward_index(const Geom& G, const Site& s, int mu)
{
    if (mu == 1) {
        if (s.xodd) return s.h;                                   // x-1 = 2 xh: same xh
        return s.xh > 0 ? s.h - 1u : s.h + G.nxh - 1u;            // x-1 = 2 (xh-1) + 1, wraps
    }
    return coord(s, mu) > 0 ? s.h - G.stride[mu] : s.h + G.stride[mu] * (G.extent[mu] - 1u);
}

// half-index of x + mu_hat
__device__ __forceinline__ uint32_t forward_index(const Geom& G, const Site& s, int mu)
{
    if (mu == 1) {
        if (!s.xodd) return s.h;                                  // x+1 = 2 xh + 1: same xh
        return s.xh + 1u < G.nxh ? s.h + 1u : s.h + 1u - G.nxh;
    }
    return coord(s, mu) + 1u < G.extent[mu] ? s.h + G.stride[mu] : s.h - G.stride[mu] * (G.extent[mu] - 1u);
}

// --------------------------------------------------------------------------------- link layout
// field[parity][mu] is a block of RECON * Vp reals (Vp = Vh rounded up to whole tiles).  Inside a block the sites
// are grouped in TILES of TW consecutive half-indices (TW = 32 for fp64, 64 for fp32); a tile stores its links
// as 16-byte chunks, chunk c of the TW sites contiguous:  block[tile][c][i],  i = h mod TW.
//   fp64: chunk = double2 = one complex entry (9 or 6 chunks of 512 bytes per tile).
//   fp32: chunk = float4 = two complex entries (RECON18: 4 chunks of 1024 bytes + the float2 tails of the tile,
//         512 bytes; RECON12: 3 chunks).
// A warp reading chunk c of 32 consecutive sites moves 512 contiguous bytes with one 128-bit load per lane, and a
// neighbour shifted by one site stays 16-byte aligned, as with chunk planes over the whole lattice; but all the
// chunks of a link for one tile now form ONE contiguous run of 32 * RECON * 8 = 4608 / 3072 bytes (the same in fp32
// with its 64-site tiles): the chunks of one link share DRAM pages, gf_pack / gf_unpack get contiguous runs on this
// side, and it is what a bulk copy moves per request (the streamed kernel of round 2, measured and removed:
// DESIGN.md section 13; a bulk copy costs ~35 ns of TMA time whatever its size).  Registers hold a link as m[18] = row-major (re, im) pairs.

template <typename T> struct Vec16;
template <> struct Vec16<double> { using type = double2; };
template <> struct Vec16<float> { using type = float4; };

template <typename T> struct Tile {
    static constexpr uint32_t W = 256u / (uint32_t)sizeof(T);      // sites per tile: 32 (fp64), 64 (fp32)
    static constexpr uint32_t SHIFT = sizeof(T) == 8 ? 5u : 6u;
};

template <typename T>
__host__ __device__ __forceinline__ uint32_t padded_vh(const Geom& G)
{
    return G.Vp[sizeof(T) == 8 ? 1 : 0];
}

// offset in reals of the block field[parity][mu]
template <typename T>
__host__ __device__ __forceinline__ size_t block_offset(uint32_t parity, int mu, int recon, const Geom& G)
{
    return (size_t)(parity * 4u + (uint32_t)mu) * (size_t)recon * (size_t)padded_vh<T>(G);
}

// 16-byte units per (link, tile): RECON * TW * sizeof(T) / 16
template <typename T, int RECON> struct TileUnits {
    static constexpr uint32_t value = (uint32_t)RECON * Tile<T>::W * (uint32_t)sizeof(T) / 16u;
};

template <int RECON>
__device__ __forceinline__ void load_link(const double* __restrict__ blk, uint32_t h, double (&m)[18])
{
    const double2* p = reinterpret_cast<const double2*>(blk) + (size_t)(h >> 5) * TileUnits<double, RECON>::value + (h & 31u);
#pragma unroll
    for (int c = 0; c < RECON / 2; ++c) {
        const double2 v = p[c * 32];
        m[2 * c] = v.x;
        m[2 * c + 1] = v.y;
    }
}

template <int RECON>
__device__ __forceinline__ void load_link(const float* __restrict__ blk, uint32_t h, float (&m)[18])
{
    const float4* p = reinterpret_cast<const float4*>(blk) + (size_t)(h >> 6) * TileUnits<float, RECON>::value + (h & 63u);
#pragma unroll
    for (int c = 0; c < RECON / 4; ++c) {
        const float4 v = p[c * 64];
        m[4 * c] = v.x;
        m[4 * c + 1] = v.y;
        m[4 * c + 2] = v.z;
        m[4 * c + 3] = v.w;
    }
    if (RECON == 18) {
        const float2 v = *(reinterpret_cast<const float2*>(p - (h & 63u) + 256) + (h & 63u));
        m[16] = v.x;
        m[17] = v.y;
    }
}

template <int RECON>
__device__ __forceinline__ void store_link(double* __restrict__ blk, uint32_t h, const double (&m)[18])
{
    double2* p = reinterpret_cast<double2*>(blk) + (size_t)(h >> 5) * TileUnits<double, RECON>::value + (h & 31u);
#pragma unroll
    for (int c = 0; c < RECON / 2; ++c) p[c * 32] = make_double2(m[2 * c], m[2 * c + 1]);
}

template <int RECON>
__device__ __forceinline__ void store_link(float* __restrict__ blk, uint32_t h, const float (&m)[18])
{
    float4* p = reinterpret_cast<float4*>(blk) + (size_t)(h >> 6) * TileUnits<float, RECON>::value + (h & 63u);
#pragma unroll
    for (int c = 0; c < RECON / 4; ++c) p[c * 64] = make_float4(m[4 * c], m[4 * c + 1], m[4 * c + 2], m[4 * c + 3]);
    if (RECON == 18) *(reinterpret_cast<float2*>(p - (h & 63u) + 256) + (h & 63u)) = make_float2(m[16], m[17]);
}

// address of the first 16-byte chunk of the link of site h (the others follow at Tile<T>::W * 16 bytes)
template <typename T, int RECON>
__device__ __forceinline__ const char* link_address(const T* blk, uint32_t h)
{
    return reinterpret_cast<const char*>(blk) +
           ((size_t)(h >> Tile<T>::SHIFT) * TileUnits<T, RECON>::value + (h & (Tile<T>::W - 1u))) * 16u;
}

// ------------------------------------------------------------------------- 3x3 complex algebra
#define GF_RE(m, a, b) (m)[2 * (3 * (a) + (b))]
#define GF_IM(m, a, b) (m)[2 * (3 * (a) + (b)) + 1]

// row 2 = conj(row 0 x row 1): the third row of an SU(3) matrix (GF_RECON12)
template <typename T>
__device__ __forceinline__ void reconstruct_row2(T (&m)[18])
{
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const int b1 = (b + 1) % 3, b2 = (b + 2) % 3;
        // (row0 x row1)_b = u0[b1] u1[b2] - u0[b2] u1[b1]
        const T re = GF_RE(m, 0, b1) * GF_RE(m, 1, b2) - GF_IM(m, 0, b1) * GF_IM(m, 1, b2)
                   - GF_RE(m, 0, b2) * GF_RE(m, 1, b1) + GF_IM(m, 0, b2) * GF_IM(m, 1, b1);
        const T im = GF_RE(m, 0, b1) * GF_IM(m, 1, b2) + GF_IM(m, 0, b1) * GF_RE(m, 1, b2)
                   - GF_RE(m, 0, b2) * GF_IM(m, 1, b1) - GF_IM(m, 0, b2) * GF_RE(m, 1, b1);
        GF_RE(m, 2, b) = re;
        GF_IM(m, 2, b) = -im;
    }
}

// the same third row, written to r[6] = (re, im) x 3 instead of into the matrix
template <typename T>
__device__ __forceinline__ void row2_of(const T (&m)[18], T (&r)[6])
{
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const int b1 = (b + 1) % 3, b2 = (b + 2) % 3;
        const T re = GF_RE(m, 0, b1) * GF_RE(m, 1, b2) - GF_IM(m, 0, b1) * GF_IM(m, 1, b2)
                   - GF_RE(m, 0, b2) * GF_RE(m, 1, b1) + GF_IM(m, 0, b2) * GF_IM(m, 1, b1);
        const T im = GF_RE(m, 0, b1) * GF_IM(m, 1, b2) + GF_IM(m, 0, b1) * GF_RE(m, 1, b2)
                   - GF_RE(m, 0, b2) * GF_IM(m, 1, b1) - GF_IM(m, 0, b2) * GF_RE(m, 1, b1);
        r[2 * b] = re;
        r[2 * b + 1] = -im;
    }
}

// Tells the compiler that v may have changed: an expression recomputed from it afterwards is not merged with
// the earlier computation (which would keep that result in registers in between).
__device__ __forceinline__ void forget(double& v) { asm volatile("" : "+d"(v)); }
__device__ __forceinline__ void forget(float& v) { asm volatile("" : "+f"(v)); }

__device__ __forceinline__ float gf_fma(float a, float b, float c) { return __fmaf_rn(a, b, c); }
__device__ __forceinline__ double gf_fma(double a, double b, double c) { return __fma_rn(a, b, c); }

// The products below are written as explicit fma chains (one multiply, then fused multiply-adds):
// two instructions per complex multiply-accumulate term instead of the three (mul, fma, add) the
// compiler emits for  re += a*b - c*d.

// out = g U, rows 0..ROWS-1 only
template <int ROWS, typename T>
__device__ __forceinline__ void mul_g_U(const T (&g)[18], const T (&U)[18], T (&out)[18])
{
#pragma unroll
    for (int a = 0; a < ROWS; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            T re = GF_RE(g, a, 0) * GF_RE(U, 0, b);
            T im = GF_RE(g, a, 0) * GF_IM(U, 0, b);
            re = gf_fma(-GF_IM(g, a, 0), GF_IM(U, 0, b), re);
            im = gf_fma(GF_IM(g, a, 0), GF_RE(U, 0, b), im);
#pragma unroll
            for (int k = 1; k < 3; ++k) {
                re = gf_fma(GF_RE(g, a, k), GF_RE(U, k, b), re);
                im = gf_fma(GF_RE(g, a, k), GF_IM(U, k, b), im);
                re = gf_fma(-GF_IM(g, a, k), GF_IM(U, k, b), re);
                im = gf_fma(GF_IM(g, a, k), GF_RE(U, k, b), im);
            }
            GF_RE(out, a, b) = re;
            GF_IM(out, a, b) = im;
        }
}

// out = U g^dagger, rows 0..ROWS-1 only:  out_ab = sum_k U_ak conj(g_bk)
template <int ROWS, typename T>
__device__ __forceinline__ void mul_U_gdag(const T (&U)[18], const T (&g)[18], T (&out)[18])
{
#pragma unroll
    for (int a = 0; a < ROWS; ++a)
#pragma unroll
        for (int b = 0; b < 3; ++b) {
            T re = GF_RE(U, a, 0) * GF_RE(g, b, 0);
            T im = GF_IM(U, a, 0) * GF_RE(g, b, 0);
            re = gf_fma(GF_IM(U, a, 0), GF_IM(g, b, 0), re);
            im = gf_fma(-GF_RE(U, a, 0), GF_IM(g, b, 0), im);
#pragma unroll
            for (int k = 1; k < 3; ++k) {
                re = gf_fma(GF_RE(U, a, k), GF_RE(g, b, k), re);
                im = gf_fma(GF_IM(U, a, k), GF_RE(g, b, k), im);
                re = gf_fma(GF_IM(U, a, k), GF_IM(g, b, k), re);
                im = gf_fma(-GF_RE(U, a, k), GF_IM(g, b, k), im);
            }
            GF_RE(out, a, b) = re;
            GF_IM(out, a, b) = im;
        }
}

__device__ __forceinline__ float gf_rsqrt(float x) { return rsqrtf(x); }
__device__ __forceinline__ double gf_rsqrt(double x) { return rsqrt(x); }

// -------------------------------------------------------------------- the SU(2) subgroup step
enum { ALGO_RELAX = 0, ALGO_OVERRELAX = 1, ALGO_STOCHASTIC = 2 };

// One of the three SU(2) maximisations of PAPER.md:76 for the subgroup (I,J).  The 2x2 block of
// K is projected on SU(2) x R+ :  Re tr[a K_sub] = a . v  for
//   a = [[a0 + i a3, a2 + i a1], [-a2 + i a1, a0 - i a3]],
//   v = (Re(K_II + K_JJ), -Im(K_IJ + K_JI), Re(K_JI - K_IJ), Im(K_JJ - K_II)),
// so eq. 9 gives a = v/|v|.  Overrelaxation (first order):
// a -> normalise(1 + omega (a - 1)) = normalise(omega v + (1 - omega)|v| e0).  Stochastic
// relaxation: a -> a^2 when `square`.
template <int I, int J, typename T>
__device__ __forceinline__ void su2_vector(const T (&K)[18], int algo, T omega, bool square, T (&a)[4])
{
    T v0 = GF_RE(K, I, I) + GF_RE(K, J, J);
    T v1 = -(GF_IM(K, I, J) + GF_IM(K, J, I));
    T v2 = GF_RE(K, J, I) - GF_RE(K, I, J);
    T v3 = GF_IM(K, J, J) - GF_IM(K, I, I);
    T nn = v0 * v0 + v1 * v1 + v2 * v2 + v3 * v3;
    a[0] = T(1);
    a[1] = a[2] = a[3] = T(0);
    if (nn > T(0)) {
        T rn = gf_rsqrt(nn);
        if (algo == ALGO_OVERRELAX) {
            const T n = nn * rn;
            v0 = omega * v0 + (T(1) - omega) * n;
            v1 *= omega;
            v2 *= omega;
            v3 *= omega;
            nn = v0 * v0 + v1 * v1 + v2 * v2 + v3 * v3;
            rn = gf_rsqrt(nn);
        }
        a[0] = v0 * rn;
        a[1] = v1 * rn;
        a[2] = v2 * rn;
        a[3] = v3 * rn;
        if (square) {
            const T t = a[0] + a[0];
            a[0] = t * a[0] - T(1);
            a[1] *= t;
            a[2] *= t;
            a[3] *= t;
        }
    }
}

// K <- E K with E the embedding of a in the subgroup (I,J):
// E_II = a0 + i a3, E_IJ = a2 + i a1, E_JI = -a2 + i a1, E_JJ = a0 - i a3
template <int I, int J, typename T>
__device__ __forceinline__ void su2_apply(T (&K)[18], const T (&a)[4])
{
#pragma unroll
    for (int b = 0; b < 3; ++b) {
        const T ir = GF_RE(K, I, b), ii = GF_IM(K, I, b), jr = GF_RE(K, J, b), ji = GF_IM(K, J, b);
        GF_RE(K, I, b) = a[0] * ir - a[3] * ii + a[2] * jr - a[1] * ji;
        GF_IM(K, I, b) = a[0] * ii + a[3] * ir + a[2] * ji + a[1] * jr;
        GF_RE(K, J, b) = -a[2] * ir - a[1] * ii + a[0] * jr + a[3] * ji;
        GF_IM(K, J, b) = -a[2] * ii + a[1] * ir + a[0] * ji - a[3] * jr;
    }
}

// (xr + i xi) (yr + i yi)
template <typename T>
__device__ __forceinline__ void cmul(T xr, T xi, T yr, T yi, T& zr, T& zi)
{
    zr = gf_fma(-xi, yi, xr * yr);
    zi = gf_fma(xi, yr, xr * yi);
}

// z += (xr + i xi) (yr + i yi)
template <typename T>
__device__ __forceinline__ void cmac(T xr, T xi, T yr, T yi, T& zr, T& zi)
{
    zr = gf_fma(-xi, yi, gf_fma(xr, yr, zr));
    zi = gf_fma(xi, yr, gf_fma(xr, yi, zi));
}

// g = E3 E2 E1 for the subgroups (0,1), (0,2), (1,2) with SU(2) vectors a, b, c, multiplied out
// using the zeros of the factors (56 instead of 144 fused multiply-adds for three dense updates
// of a matrix that starts as the identity).
template <typename T>
__device__ __forceinline__ void compose_g(const T (&a)[4], const T (&b)[4], const T (&c)[4], T (&g)[18])
{
    // after E1: row0 = (p, q, 0), row1 = (r, s, 0), row2 = (0, 0, 1)
    const T pr = a[0], pi = a[3], qr = a[2], qi = a[1], rr = -a[2], ri = a[1], sr = a[0], si = -a[3];
    // E2 on rows (0,2): row0' = P row0 + Q row2 = (P p, P q, Q);  row2' = R row0 + S row2 = (R p, R q, S)
    const T Pr = b[0], Pi = b[3], Qr = b[2], Qi = b[1], Rr = -b[2], Ri = b[1], Sr = b[0], Si = -b[3];
    cmul(Pr, Pi, pr, pi, GF_RE(g, 0, 0), GF_IM(g, 0, 0));
    cmul(Pr, Pi, qr, qi, GF_RE(g, 0, 1), GF_IM(g, 0, 1));
    GF_RE(g, 0, 2) = Qr;
    GF_IM(g, 0, 2) = Qi;
    T x0r, x0i, x1r, x1i;            // row2' entries 0, 1 (entry 2 is S)
    cmul(Rr, Ri, pr, pi, x0r, x0i);
    cmul(Rr, Ri, qr, qi, x1r, x1i);
    // E3 on rows (1,2): row1'' = P3 row1 + Q3 row2';  row2'' = R3 row1 + S3 row2'
    const T P3r = c[0], P3i = c[3], Q3r = c[2], Q3i = c[1], R3r = -c[2], R3i = c[1], S3r = c[0], S3i = -c[3];
    cmul(P3r, P3i, rr, ri, GF_RE(g, 1, 0), GF_IM(g, 1, 0));
    cmac(Q3r, Q3i, x0r, x0i, GF_RE(g, 1, 0), GF_IM(g, 1, 0));
    cmul(P3r, P3i, sr, si, GF_RE(g, 1, 1), GF_IM(g, 1, 1));
    cmac(Q3r, Q3i, x1r, x1i, GF_RE(g, 1, 1), GF_IM(g, 1, 1));
    cmul(Q3r, Q3i, Sr, Si, GF_RE(g, 1, 2), GF_IM(g, 1, 2));
    cmul(R3r, R3i, rr, ri, GF_RE(g, 2, 0), GF_IM(g, 2, 0));
    cmac(S3r, S3i, x0r, x0i, GF_RE(g, 2, 0), GF_IM(g, 2, 0));
    cmul(R3r, R3i, sr, si, GF_RE(g, 2, 1), GF_IM(g, 2, 1));
    cmac(S3r, S3i, x1r, x1i, GF_RE(g, 2, 1), GF_IM(g, 2, 1));
    cmul(S3r, S3i, Sr, Si, GF_RE(g, 2, 2), GF_IM(g, 2, 2));
}

// a4: the local maximiser g(x) = E3 E2 E1 of Re tr[g K] over the three SU(2) subgroups in the
// order (0,1), (0,2), (1,2), K refreshed between the steps.  K is destroyed.
template <typename T>
__device__ __forceinline__ void solve_site(T (&K)[18], int algo, T omega, bool sq0, bool sq1, bool sq2, T (&g)[18])
{
    T a[4], b[4], c[4];
    su2_vector<0, 1>(K, algo, omega, sq0, a);
    su2_apply<0, 1>(K, a);
    su2_vector<0, 2>(K, algo, omega, sq1, b);
    su2_apply<0, 2>(K, b);
    su2_vector<1, 2>(K, algo, omega, sq2, c);
    compose_g(a, b, c, g);
}

// --------------------------------------------------------------------------- Philox4x32-10
// Salmon et al., SC'11 (public algorithm).  Counter-based: no state in memory.
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&out)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

}  // namespace gf
