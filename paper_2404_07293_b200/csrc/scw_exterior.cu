// Exterior field: eq. 9 in the half-spaces above and below the sample.
//   above:  p(s_m, z) = p_inc_m G[s_z(n), z_inc, z] + p_face_m G[-s_z(n), z_face, z]
//   below:  p(s_m, z) = p_face_m G[s_z(n), z_face, z]
// s_z(n) = sqrt(n^2 - |s_m|^2) on the Im >= 0 branch (eq. 2), s_m = lambda (u/X, v/Y) (eq. 6),
// G(A, z_a, z_b) = exp[ik (z_b - z_a) A] (eq. 7).  The reflected wave carries -s_z (reading c-17).
// k_exterior_spectra evaluates eq. 9 on z planes (its output feeds the separable synthesis, eq. 10);
// k_exterior_modes tabulates the same waves as a plane-wave list for the direct point kernels.
#include "scw_internal.h"
#include "scw_exterior.cuh"

namespace scw {

template <typename T2>
__global__ void k_exterior_spectra(int U, int Vn, double lam_over_X, double lam_over_Y, double inv_lambda, int side,
                                   double n_re, double n_im, double z_face, double z_inc, const T2* __restrict__ p_face,
                                   const T2* __restrict__ p_inc, int64_t Fz, const double* __restrict__ z,
                                   T2* __restrict__ P, int64_t ldP)
{
    const int M = U * Vn;
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;      // (plane i, frequency m), m fastest
    if (idx >= (int64_t)M * Fz) return;
    const int64_t i = idx / M;
    const int m = (int)(idx - i * M);
    double sx, sy;
    ext_freq(U, Vn, m, lam_over_X, lam_over_Y, sx, sy);
    const double2 sz = ext_sz(n_re, n_im, sx, sy);
    const double zi = z[i];
    // face wave: transmitted (+s_z) below, reflected (-s_z) above
    const double2 gf = side == SCW_SIDE_BELOW ? sz : make_double2(-sz.x, -sz.y);
    const double2 wf = ext_green(gf, (zi - z_face) * inv_lambda);
    double2 wi = make_double2(0.0, 0.0);
    const bool inc = side == SCW_SIDE_ABOVE && p_inc != nullptr;
    if (inc) wi = ext_green(sz, (zi - z_inc) * inv_lambda);
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) {
        const T2 a = p_face[3 * m + comp];
        double er = (double)a.x * wf.x - (double)a.y * wf.y;
        double ei = (double)a.x * wf.y + (double)a.y * wf.x;
        if (inc) {
            const T2 b = p_inc[3 * m + comp];
            er += (double)b.x * wi.x - (double)b.y * wi.y;
            ei += (double)b.x * wi.y + (double)b.y * wi.x;
        }
        T2 o;
        o.x = (decltype(o.x))er;
        o.y = (decltype(o.y))ei;
        P[i * ldP + (int64_t)comp * M + m] = o;
    }
}

void launch_exterior_spectra(scw_ctx* ctx, const scw_exterior* e, int64_t Fz, const double* z, void* P, int64_t ldP)
{
    const int64_t n = (int64_t)e->U * e->Vn * Fz;
    const unsigned blocks = (unsigned)((n + 255) / 256);
    KernelScope ks(ctx, KC_EXTERIOR);
    if (e->dtype == SCW_C64)
        k_exterior_spectra<float2><<<blocks, 256, 0, ctx->stream>>>(
            e->U, e->Vn, e->lambda / e->X, e->lambda / e->Y, 1.0 / e->lambda, e->side, e->n_re, e->n_im, e->z_face, e->z_inc,
            (const float2*)e->p_face, (const float2*)e->p_inc, Fz, z, (float2*)P, ldP);
    else
        k_exterior_spectra<double2><<<blocks, 256, 0, ctx->stream>>>(
            e->U, e->Vn, e->lambda / e->X, e->lambda / e->Y, 1.0 / e->lambda, e->side, e->n_re, e->n_im, e->z_face, e->z_inc,
            (const double2*)e->p_face, (const double2*)e->p_inc, Fz, z, (double2*)P, ldP);
}

// Plane-wave list of the half-space: wave j < M is the face wave of frequency j, wave M + m the incident wave.
template <typename T2>
__global__ void k_exterior_modes(int U, int Vn, double lam_over_X, double lam_over_Y, int side, double n_re, double n_im,
                                 double z_face, double z_inc, const T2* __restrict__ p_face, const T2* __restrict__ p_inc,
                                 int64_t J, double* __restrict__ sx_out, double* __restrict__ sy_out,
                                 double2* __restrict__ gamma, double* __restrict__ zref, T2* __restrict__ p)
{
    const int M = U * Vn;
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= J) return;
    const bool incident = j >= M;
    const int m = (int)(incident ? j - M : j);
    double sx, sy;
    ext_freq(U, Vn, m, lam_over_X, lam_over_Y, sx, sy);
    const double2 sz = ext_sz(n_re, n_im, sx, sy);
    const bool minus = !incident && side == SCW_SIDE_ABOVE;                  // reflected wave
    sx_out[j] = sx;
    sy_out[j] = sy;
    gamma[j] = minus ? make_double2(-sz.x, -sz.y) : sz;
    zref[j] = incident ? z_inc : z_face;
    const T2* src = incident ? p_inc : p_face;
#pragma unroll
    for (int comp = 0; comp < 3; ++comp) p[3 * j + comp] = src[3 * m + comp];
}

static int64_t exterior_waves(const scw_exterior* e)
{
    const int64_t M = (int64_t)e->U * e->Vn;
    return (e->side == SCW_SIDE_ABOVE && e->p_inc) ? 2 * M : M;
}

size_t exterior_points_bytes(const scw_exterior* e)
{
    const int64_t J = exterior_waves(e);
    const size_t es = e->dtype == SCW_C64 ? 8 : 16;
    return 3 * align_up((size_t)J * 8) + align_up((size_t)J * 16) + align_up((size_t)J * 3 * es) + points_table_bytes(e->dtype, J);
}

void launch_exterior_points(scw_ctx* ctx, const scw_exterior* e, int64_t N, const double* r, void* E, void* ws)
{
    const int64_t J = exterior_waves(e);
    const size_t es = e->dtype == SCW_C64 ? 8 : 16;
    Carver cv(ws);
    double* sx = (double*)cv.take((size_t)J * 8);
    double* sy = (double*)cv.take((size_t)J * 8);
    double* zref = (double*)cv.take((size_t)J * 8);
    double2* gamma = (double2*)cv.take((size_t)J * 16);
    void* p = cv.take((size_t)J * 3 * es);
    void* table = cv.take(points_table_bytes(e->dtype, J));
    {
        KernelScope ks(ctx, KC_EXTERIOR);
        const unsigned blocks = (unsigned)((J + 127) / 128);
        if (e->dtype == SCW_C64)
            k_exterior_modes<float2><<<blocks, 128, 0, ctx->stream>>>(
                e->U, e->Vn, e->lambda / e->X, e->lambda / e->Y, e->side, e->n_re, e->n_im, e->z_face, e->z_inc,
                (const float2*)e->p_face, (const float2*)e->p_inc, J, sx, sy, gamma, zref, (float2*)p);
        else
            k_exterior_modes<double2><<<blocks, 128, 0, ctx->stream>>>(
                e->U, e->Vn, e->lambda / e->X, e->lambda / e->Y, e->side, e->n_re, e->n_im, e->z_face, e->z_inc,
                (const double2*)e->p_face, (const double2*)e->p_inc, J, sx, sy, gamma, zref, (double2*)p);
    }
    scw_modes m = {};
    m.struct_size = sizeof(scw_modes);
    m.kind = SCW_MODES_PLANEWAVE;
    m.dtype = e->dtype;
    m.J = J;
    m.lambda = e->lambda;
    m.sx = sx;
    m.sy = sy;
    m.gamma = reinterpret_cast<const double*>(gamma);
    m.zref = zref;
    m.p = p;
    launch_points_planewave(ctx, &m, N, r, E, table);
}

}  // namespace scw
