// Plane kernel for (y,z) planes that do not fit, or fit only once, in one SM's shared memory (128 x 128: 262 KB; 96 x 100 and
// 108 x 108: 170 / 188 KB, i.e. one CTA per SM and nothing to overlap its phases with): a thread-block CLUSTER of two CTAs holds the
// plane, rows [h*NY/2, (h+1)*NY/2) in CTA h, and the one stage that couples the two halves reads and writes the partner's rows
// through distributed shared memory (mapa + ld/st.shared::cluster).
//
// Same transform, orders and functors as plane_kernel (fft_fused.cuh): forward = decimation in frequency,
//   z stage R1z, z stage R2z            on the CTA's own rows
//   y stage R1y (rows i + R2y*r)        r < R1y/2 lives in CTA 0, r >= R1y/2 in CTA 1: CTA h does the columns of its half of z
//   y stage R2y (blocks of R2y rows)    own rows again, straight to global memory
// and the inverse runs the stages backwards.  Two cluster barriers per unit around the coupled stage.
#pragma once
#include <cooperative_groups.h>
#include "fft_fused.cuh"

namespace tddft {

__device__ __forceinline__ unsigned map_to_rank(unsigned smem_addr, unsigned rank) {
    unsigned r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(smem_addr), "r"(rank));
    return r;
}
__device__ __forceinline__ cplx ld_cluster(unsigned addr) {
    cplx v;
    asm volatile("ld.shared::cluster.v2.f64 {%0, %1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr) : "memory");
    return v;
}
__device__ __forceinline__ void st_cluster(unsigned addr, cplx v) {
    asm volatile("st.shared::cluster.v2.f64 [%0], {%1, %2};" ::"r"(addr), "d"(v.x), "d"(v.y) : "memory");
}

template <int NY, int NZ, int NTHR, int MINB, bool INV, class Load, class Store>
__global__ void __launch_bounds__(NTHR, MINB) plane_cluster_kernel(Load ld, Store st, int nx, int nunits, const cplx* __restrict__ twy_g, const cplx* __restrict__ twz_g) {
    namespace cg = cooperative_groups;
    using TY = Two<NY>; using TZ = Two<NZ>;
    constexpr int R1y = TY::R1, R2y = TY::R2, R1z = TZ::R1, R2z = TZ::R2;
    constexpr int PITCH = TZ::PITCH, HY = NY / 2, HZ = NZ / 2;
    static_assert(R1y % 2 == 0 && NZ % 2 == 0, "the coupled stage splits the rows r < R1y/2 | r >= R1y/2 and the columns in halves");
    extern __shared__ cplx sm[];
    cg::cluster_group cluster = cg::this_cluster();
    const unsigned h = cluster.block_rank();
    const int tid = threadIdx.x;
    pdl_launch_dependents();
    const unsigned sm_local = (unsigned)__cvta_generic_to_shared(sm);
    const unsigned sm_rank[2] = {map_to_rank(sm_local, 0), map_to_rank(sm_local, 1)};
    typedef decltype(bind(ld, 0, 0, 0L)) BL;
    typedef typename BL::Raw Raw;
    const int nbatch = nunits / nx;
    const int ncl = gridDim.x / 2, cl = blockIdx.x / 2;
    pdl_wait();
    for (int u = cl; u < nunits; u += ncl) {
        const int xpl = u / nbatch, b = u - xpl * nbatch;
        BL L = bind(ld, b, xpl, (long)xpl * NY * NZ);
        const auto S = bind(st, b, xpl, (long)xpl * NY * NZ);
        {   // operands of the unit this cluster takes next -> L2 (each CTA its half of the threads' share; no registers held)
            const int un = u + ncl;
            if (un < nunits) { const int xn = un / nbatch, bn = un - xn * nbatch; bind(ld, bn, xn, (long)xn * NY * NZ).prefetch_l2(NY * NZ, tid + (int)h * NTHR, 2 * NTHR); }
        }
        if constexpr (!INV) {
            // z stage 1 on the own rows: global -> registers -> shared
            auto z1 = [&](auto mode_) {
                constexpr int MD = decltype(mode_)::value;
                for (int t = tid; t < HY * R2z; t += NTHR) {
                    const int yl = t / R2z, i = t - yl * R2z, y = (int)h * HY + yl;
                    cplx x[R1z];
#pragma unroll
                    for (int r = 0; r < R1z; ++r) { const Raw q = L.template fetch<MD>(y * NZ + i + R2z * r); x[r] = L.make(q); }
                    Dft<R1z, false>::run(x);
                    cplx* row = sm + yl * PITCH;
                    row[TZ::pad(i)] = x[0];
#pragma unroll
                    for (int k = 1; k < R1z; ++k) row[TZ::pad(i + R2z * k)] = cmul(x[k], __ldg(twz_g + i * k));
                }
            };
            if (BL::kModes > 1 && L.mode() == 1) z1(IC<1>{}); else z1(IC<0>{});
            __syncthreads();
            for (int t = tid; t < HY * R1z; t += NTHR) {      // z stage 2, in place
                const int yl = t / R1z, k1 = t - yl * R1z;
                cplx* blk = sm + yl * PITCH + TZ::pad(k1 * R2z);
                cplx x[R2z];
#pragma unroll
                for (int i = 0; i < R2z; ++i) x[i] = blk[i];
                Dft<R2z, false>::run(x);
#pragma unroll
                for (int i = 0; i < R2z; ++i) blk[i] = x[i];
            }
            cluster.sync();
            // y stage 1 on the columns of this CTA's half of z: rows i + R2y*r, half of them in the partner's shared memory
            for (int t = tid; t < HZ * R2y; t += NTHR) {
                const int zl = t / R2y, i = t - zl * R2y, zp = (int)h * HZ + zl;
                const unsigned off = (unsigned)((TZ::pad(zp) + i * PITCH) * sizeof(cplx));
                cplx x[R1y];
#pragma unroll
                for (int r = 0; r < R1y; ++r) x[r] = ld_cluster(sm_rank[r >= R1y / 2] + off + (unsigned)(((r % (R1y / 2)) * R2y * PITCH) * sizeof(cplx)));
                Dft<R1y, false>::run(x);
#pragma unroll
                for (int k = 0; k < R1y; ++k) {
                    const cplx v = k == 0 ? x[0] : cmul(x[k], __ldg(twy_g + i * k));
                    st_cluster(sm_rank[k >= R1y / 2] + off + (unsigned)(((k % (R1y / 2)) * R2y * PITCH) * sizeof(cplx)), v);
                }
            }
            cluster.sync();
            // y stage 2 on the own rows (blocks k1 of R2y rows): shared -> registers -> global
            for (int t = tid; t < NZ * (R1y / 2); t += NTHR) {
                const int k1l = t / NZ, zp = t - k1l * NZ;
                const cplx* col = sm + TZ::pad(zp) + (k1l * R2y) * PITCH;
                cplx x[R2y];
#pragma unroll
                for (int i = 0; i < R2y; ++i) x[i] = col[i * PITCH];
                Dft<R2y, false>::run(x);
                const int k1 = (int)h * (R1y / 2) + k1l;
#pragma unroll
                for (int k = 0; k < R2y; ++k) S((k1 * R2y + k) * NZ + zp, x[k]);
            }
            __syncthreads();      // the own rows are rewritten by the next unit's z stage 1
        } else {
            // y inverse stage R2y on the own row blocks: global -> registers -> shared
            for (int t = tid; t < NZ * (R1y / 2); t += NTHR) {
                const int k1l = t / NZ, zp = t - k1l * NZ, k1 = (int)h * (R1y / 2) + k1l;
                cplx x[R2y];
#pragma unroll
                for (int i = 0; i < R2y; ++i) { const Raw q = L.template fetch<0>((k1 * R2y + i) * NZ + zp); x[i] = L.make(q); }
                Dft<R2y, true>::run(x);
                cplx* col = sm + TZ::pad(zp) + (k1l * R2y) * PITCH;
#pragma unroll
                for (int i = 0; i < R2y; ++i) col[i * PITCH] = x[i];
            }
            cluster.sync();
            // y inverse stage R1y (conjugate twiddle before the butterfly) on the columns of this CTA's half of z
            for (int t = tid; t < HZ * R2y; t += NTHR) {
                const int zl = t / R2y, i = t - zl * R2y, zp = (int)h * HZ + zl;
                const unsigned off = (unsigned)((TZ::pad(zp) + i * PITCH) * sizeof(cplx));
                cplx x[R1y];
#pragma unroll
                for (int k = 0; k < R1y; ++k) {
                    const cplx v = ld_cluster(sm_rank[k >= R1y / 2] + off + (unsigned)(((k % (R1y / 2)) * R2y * PITCH) * sizeof(cplx)));
                    x[k] = k == 0 ? v : cmulc(v, __ldg(twy_g + i * k));
                }
                Dft<R1y, true>::run(x);
#pragma unroll
                for (int r = 0; r < R1y; ++r) st_cluster(sm_rank[r >= R1y / 2] + off + (unsigned)(((r % (R1y / 2)) * R2y * PITCH) * sizeof(cplx)), x[r]);
            }
            cluster.sync();
            for (int t = tid; t < HY * R1z; t += NTHR) {      // z inverse stage R2z on the own rows, in place
                const int yl = t / R1z, k1 = t - yl * R1z;
                cplx* blk = sm + yl * PITCH + TZ::pad(k1 * R2z);
                cplx x[R2z];
#pragma unroll
                for (int i = 0; i < R2z; ++i) x[i] = blk[i];
                Dft<R2z, true>::run(x);
#pragma unroll
                for (int i = 0; i < R2z; ++i) blk[i] = x[i];
            }
            __syncthreads();
            for (int t = tid; t < HY * R2z; t += NTHR) {      // z inverse stage R1z: shared -> registers -> global (natural order)
                const int yl = t / R2z, i = t - yl * R2z, y = (int)h * HY + yl;
                const cplx* row = sm + yl * PITCH;
                cplx x[R1z];
                x[0] = row[TZ::pad(i)];
#pragma unroll
                for (int k = 1; k < R1z; ++k) x[k] = cmulc(row[TZ::pad(i + R2z * k)], __ldg(twz_g + i * k));
                Dft<R1z, true>::run(x);
#pragma unroll
                for (int r = 0; r < R1z; ++r) S(y * NZ + i + R2z * r, x[r]);
            }
            // the partner's coupled stage of the NEXT unit writes these rows only after the next unit's first cluster barrier,
            // which this CTA reaches after it has finished the stores above
            __syncthreads();
        }
    }
    cluster.sync();      // no CTA exits while its partner may still address its shared memory
}

}  // namespace tddft
