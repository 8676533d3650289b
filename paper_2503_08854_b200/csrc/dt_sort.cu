// dt_sort.cu -- sky order: the orbits of a work unit are processed in the order of where they are on the sky.
//
// Kernels 1 and 3 decide per WARP: a warp refines an exposure when ANY of its 32 orbits may be near it, the group
// ephemeris gate removes an exposure when NONE can be, and the 32 lanes of a warp gather from wherever their orbits
// land.  How much a warp has to do therefore depends on how alike its 32 orbits are -- i.e. on the order the caller
// happened to list them in (NS subsystem 3 asks for hits binned "for L2 and coalesced locality"; PAPER.md:346 names the
// "reorganization" of the search for reuse as the open problem).  Here each unit of up to 2^20 orbits is re-ordered
// before kernel 1: one Kepler solve per orbit at the survey's middle exposure gives its apparent direction from the
// observer, the direction is binned into equal-area cells (512 bands in sin(dec) x 2048 in RA, 0.2 deg across), and
// the orbits are sorted by cell with a stable radix sort (deterministic: same input, same order).  Kernels 1 and 3 run
// on the sorted copy; the per-orbit sums are scattered back to the caller's order before the SNR is formed, so
// nothing outside this file sees the permutation.  Orbits that belong together (the members of a family around a
// known object, neighbouring nodes of a search grid) end up in the same warps whatever order they came in.
//
// The sort itself is library code (CUB's DeviceRadixSort, 21-bit keys, ~0.1 ms per unit against milliseconds of
// kernel 1): it orders work, it computes nothing of the method.
#include <cub/device/device_radix_sort.cuh>

#include "dt_common.cuh"
#include "dt_orbit.cuh"

namespace dt {

namespace {

constexpr int kSortThreads = 256;
constexpr int kBandBits = 9, kRaBits = 11;          // 512 x 2048 equal-area cells
constexpr int kKeyBits = kBandBits + kRaBits + 1;    // + 1: orbits with a perihelion inside kLoosePerihelion sort last
// The group ephemeris gate of kernel 1 decides per warp and needs every lane's remainder bound to be tight; the bound grows
// like 1 / r^3, so ONE orbit that comes close to the Sun switches the gate off for its 31 neighbours.  Orbits whose
// perihelion lies inside 0.7 AU are therefore kept apart from the others (only the near-Earth config has any).
constexpr double kLoosePerihelion = 0.7;

// apparent direction (geometric, no light-time: a sort key, not a result) at the key exposure -> cell index
__global__ void __launch_bounds__(kSortThreads) k_sky_keys(const double *__restrict__ elements,
                                                          const double *__restrict__ t0_orbit, int64_t n, double t0,
                                                          const ExpRec *key_exp, double gm, double cos_eps,
                                                          double sin_eps, uint32_t *__restrict__ keys,
                                                          uint32_t *__restrict__ index)
{
    const int64_t i = (int64_t)blockIdx.x * kSortThreads + threadIdx.x;
    const int64_t ic = min(i, n - 1);                   // whole warps call the (warp-voting) Kepler solve
    double el[6];
#pragma unroll
    for (int k = 0; k < 6; ++k) el[k] = elements[ic * 6 + k];
    const double te = t0_orbit ? t0_orbit[ic] : t0;
    const Orbit o = orbit_setup(el, gm, cos_eps, sin_eps, 0.0, 0.0);
    const ExpRec x = *key_exp;
    const double M = fma(o.n, x.t - te, o.M0);
    const Kepler K = kepler_cold(o.e, isfinite(M) ? M : 0.0);
    const double X0 = K.c - o.e;
    const double qx = fma(o.Ax, X0, fma(o.Bx, K.s, -x.Rx));
    const double qy = fma(o.Ay, X0, fma(o.By, K.s, -x.Ry));
    const double qz = fma(o.Az, X0, fma(o.Bz, K.s, -x.Rz));
    const double rho = sqrt(fma(qx, qx, fma(qy, qy, qz * qz)));
    uint32_t key = (1u << kKeyBits) - 1u;               // invalid orbits, degenerate directions: last
    if (o.valid && isfinite(te) && rho > 0.0 && isfinite(rho)) {
        const double z = fmin(fmax(qz / rho, -1.0), 1.0);
        double ra = atan2(qy, qx) * kInvTwoPi;          // (-0.5, 0.5]
        if (ra < 0.0) ra += 1.0;
        const uint32_t band = min((uint32_t)((z + 1.0) * 0.5 * (double)(1 << kBandBits)), (1u << kBandBits) - 1u);
        const uint32_t cell = min((uint32_t)(ra * (double)(1 << kRaBits)), (1u << kRaBits) - 1u);
        key = (band << kRaBits) | cell;
        if (el[0] * (1.0 - el[1]) < kLoosePerihelion) key |= 1u << (kBandBits + kRaBits);
    }
    if (i < n) {
        keys[i] = key;
        index[i] = (uint32_t)i;
    }
}

// sorted copy: row i of the sorted elements is row perm[i] of the caller's (48-B rows as three 16-B pieces)
__global__ void __launch_bounds__(kSortThreads) k_permute_rows(const double *__restrict__ elements,
                                                              const double *__restrict__ t0_orbit,
                                                              const uint32_t *__restrict__ perm, int64_t n,
                                                              double *__restrict__ elements_sorted,
                                                              double *__restrict__ t0_sorted)
{
    const int64_t k = (int64_t)blockIdx.x * kSortThreads + threadIdx.x;
    if (k >= n * 3) return;
    const int64_t i = k / 3, part = k - i * 3;
    const int64_t src = perm[i];
    if ((reinterpret_cast<uintptr_t>(elements) & 15u) == 0) {
        reinterpret_cast<double2 *>(elements_sorted)[k] = reinterpret_cast<const double2 *>(elements)[src * 3 + part];
    } else {
        elements_sorted[2 * k] = elements[src * 6 + 2 * part];
        elements_sorted[2 * k + 1] = elements[src * 6 + 2 * part + 1];
    }
    if (t0_sorted && part == 0) t0_sorted[i] = t0_orbit[src];
}

// the per-orbit sums back into the caller's order
__global__ void __launch_bounds__(kSortThreads) k_unpermute_sums(const uint32_t *__restrict__ perm, int64_t n,
                                                                int64_t unit, const double *__restrict__ S_s,
                                                                const double *__restrict__ Wt_s,
                                                                const int32_t *__restrict__ cnt_s, double *__restrict__ S,
                                                                double *__restrict__ Wt, int32_t *__restrict__ cnt)
{
    const int64_t i = (int64_t)blockIdx.x * kSortThreads + threadIdx.x;
    if (i >= n) return;
    const int64_t o0 = i / unit * unit;                 // the permutation is local to the orbit unit
    const int64_t dst = o0 + perm[i];
    S[dst] = S_s[i];
    Wt[dst] = Wt_s[i];
    cnt[dst] = cnt_s[i];
}

}  // namespace

size_t sky_sort_temp_bytes(int64_t n_max)
{
    size_t bytes = 0;
    cub::DeviceRadixSort::SortPairs(nullptr, bytes, (const uint32_t *)nullptr, (uint32_t *)nullptr,
                                    (const uint32_t *)nullptr, (uint32_t *)nullptr, (int)n_max, 0, kKeyBits);
    return bytes;
}

// One unit (n <= 2^31 orbits): perm [n], and the sorted copies of the elements (and epochs, when given).
// keys_in / keys_out / index_in: scratch [n] uint32 each; temp: sky_sort_temp_bytes(n) bytes.
cudaError_t sky_sort_unit(const double *elements, const double *t0_orbit, int64_t n, double t0, const ExpRec *key_exp,
                          double gm, double cos_eps, double sin_eps, uint32_t *keys_in, uint32_t *keys_out,
                          uint32_t *index_in, void *temp, size_t temp_bytes, uint32_t *perm, double *elements_sorted,
                          double *t0_sorted, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    k_sky_keys<<<(unsigned)((n + kSortThreads - 1) / kSortThreads), kSortThreads, 0, stream>>>(
        elements, t0_orbit, n, t0, key_exp, gm, cos_eps, sin_eps, keys_in, index_in);
    cudaError_t e = cub::DeviceRadixSort::SortPairs(temp, temp_bytes, (const uint32_t *)keys_in, keys_out,
                                                    (const uint32_t *)index_in, perm, (int)n, 0, kKeyBits, stream);
    if (e != cudaSuccess) return e;
    if (elements_sorted)
        k_permute_rows<<<(unsigned)((n * 3 + kSortThreads - 1) / kSortThreads), kSortThreads, 0, stream>>>(
            elements, t0_orbit, perm, n, elements_sorted, t0_orbit ? t0_sorted : nullptr);
    return cudaGetLastError();
}

cudaError_t sky_unsort_sums(const uint32_t *perm, int64_t n, int64_t unit, const double *S_s, const double *Wt_s,
                            const int32_t *cnt_s, double *S, double *Wt, int32_t *cnt, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    k_unpermute_sums<<<(unsigned)((n + kSortThreads - 1) / kSortThreads), kSortThreads, 0, stream>>>(perm, n, unit, S_s,
                                                                                                  Wt_s, cnt_s, S, Wt, cnt);
    return cudaGetLastError();
}

}  // namespace dt
