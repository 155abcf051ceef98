// radt_setup.cu -- K1 ray geometry, per-call tables, field packing, gradient unpacking, L2 loss.
// One fused "setup" launch precedes every march so that small problems stay launch-lean.
#include "radt_dev.cuh"
#include "radt_kernels.h"

// ---------------------------------------------------------------------------------------------
// K1 ray geometry (O1-O3): per pixel the clipped interval {s0, ds}; ds = 0 marks a miss.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ RayRec clip_ray(const DevGeom &G, const DevGrid &g, int nx, int ny, int nstep, int ix, int iy)
{
    double ox, oy, oz, X, Y;
    pixel_origin(G, nx, ny, ix, iy, ox, oy, oz, X, Y);
    RayRec rr;
    rr.s0 = 0.0; rr.ds = 0.0; rr.k_lo = 0; rr.k_hi = 0; rr.pad0 = 0; rr.pad1 = 0;
    if (g.kind == 0) {
        // s = 0 is the closest approach to the star, |p(s)|^2 = b^2 + s^2
        double b2 = X * X + Y * Y;
        if (!(b2 < g.rb2)) return rr;
        double sh = sqrt(g.rb2 - b2);
        rr.s0 = -sh;
        rr.ds = 2.0 * sh / (double)nstep;
        // Conservative s-interval that contains every in-grid sample: inside the cylinder r <= r_max and, for a
        // wedge symmetric about the midplane seen from outside its opening angle, between the two cones
        // |z| <= zeta_hi r.  Each is a quadratic inequality in s.  One step of slack on both sides.
        double sa = rr.s0, sb = -rr.s0;
        double a = G.wx * G.wx + G.wy * G.wy, bq = ox * G.wx + oy * G.wy, c = ox * ox + oy * oy;
        bool empty = false;
        if (a > 1e-14) {
            double disc = bq * bq - a * (c - g.rmax2);
            if (disc < 0.0) empty = true;
            else { double sq = sqrt(disc); sa = fmax(sa, (-bq - sq) / a); sb = fmin(sb, (-bq + sq) / a); }
        } else if (c > g.rmax2) {
            empty = true;
        }
        bool wedge = (g.mirror && g.zlo == 0.0) || (!g.mirror && g.zlo == -g.zhi);
        if (wedge && !empty) {
            double z2 = g.zhi * g.zhi;
            double A = G.wz * G.wz - z2 * a, B = oz * G.wz - z2 * bq, C = oz * oz - z2 * c;   // A s^2 + 2 B s + C <= 0
            if (A > 1e-12) {
                double disc = B * B - A * C;
                if (disc < 0.0) empty = true;
                else { double sq = sqrt(disc); sa = fmax(sa, (-B - sq) / A); sb = fmin(sb, (-B + sq) / A); }
            }
        }
        if (!empty && sb >= sa) {
            double klo = floor((sa - rr.s0) / rr.ds - 0.5) - 1.0, khi = ceil((sb - rr.s0) / rr.ds - 0.5) + 2.0;
            rr.k_lo = (int)fmin(fmax(klo, 0.0), (double)nstep);
            rr.k_hi = (int)fmin(fmax(khi, 0.0), (double)nstep);
        }
        return rr;
    }
    if (g.kind == 2) {
        // spherical grid: bounding sphere of radius r_max; every step may lie inside
        double b2 = X * X + Y * Y;
        if (!(b2 < g.rb2)) return rr;
        double sh = sqrt(g.rb2 - b2);
        rr.s0 = -sh;
        rr.ds = 2.0 * sh / (double)nstep;
        rr.k_lo = 0; rr.k_hi = nstep;
        return rr;
    }
    const double o[3] = { ox, oy, oz }, d[3] = { G.wx, G.wy, G.wz };
    double tmin = -INFINITY, tmax = INFINITY;
#pragma unroll
    for (int a = 0; a < 3; ++a) {
        if (d[a] != 0.0) {
            double t1 = (g.lo[a] - o[a]) / d[a], t2 = (g.hi[a] - o[a]) / d[a];
            tmin = fmax(tmin, fmin(t1, t2));
            tmax = fmin(tmax, fmax(t1, t2));
        } else if (o[a] < g.lo[a] || o[a] > g.hi[a]) {
            return rr;
        }
    }
    if (!(tmax > tmin)) return rr;
    rr.s0 = tmin;
    rr.ds = (tmax - tmin) / (double)nstep;
    rr.k_lo = 0; rr.k_hi = nstep;
    return rr;
}

// Block roles: [0, nb_rays) rays; then nb_tab blocks of tables; then nb_occ blocks of occupancy words; the rest
// pack fields.
__global__ void __launch_bounds__(256) k_setup(const __grid_constant__ SetupParams P, const __grid_constant__ LevelTable L,
                                               const __grid_constant__ ChanTable V, int nb_rays, int nb_tab, int nb_occ)
{
    int blk = blockIdx.x;
    if (blk < nb_rays) {
        long long per_item = (long long)P.nx * P.ny;
        long long q = (long long)blk * blockDim.x + threadIdx.x;
        if (q >= per_item * P.nbatch) return;
        int b = (int)(q / per_item);
        long long rem = q - (long long)b * per_item;
        int iy = (int)(rem / P.nx), ix = (int)(rem - (long long)iy * P.nx);
        RayRec rr = clip_ray(P.geom[b], P.grid, P.nx, P.ny, P.nstep, ix, iy);
        long long dst = (long long)(P.b0 + b) * per_item + rem;
        if (P.ws.rays) P.ws.rays[dst] = rr;
        if (P.rays_user) P.rays_user[dst] = make_double2(rr.s0, rr.ds);
        return;
    }
    blk -= nb_rays;
    if (blk < nb_tab) {
        int t = blk * blockDim.x + threadIdx.x;
        {
            // partition function Q(T) = sum g_J exp(-E_J/T) and dQ/dlnT on a log2-T lattice: one warp
            // per entry, lanes over levels (a per-thread loop over the levels was a 41-deep chain of fp64 exp and
            // the longest pole of the launch)
            int e = t >> 5, ln = t & 31;
            if (e <= RADT_NQ + 1) {
                double T = exp2((double)e * (double)RADT_NQ_OCTAVES / (double)RADT_NQ);
                double q = 0.0, dq = 0.0;
                for (int l = ln; l < P.nlev; l += 32) {
                    double y = L.e[l] / T;
                    double w = L.g[l] * exp(-y);
                    q += w;
                    dq += w * y;
                }
#pragma unroll
                for (int m = 16; m > 0; m >>= 1) {
                    q += __shfl_xor_sync(0xffffffffu, q, m);
                    dq += __shfl_xor_sync(0xffffffffu, dq, m);
                }
                if (ln == 0) P.ws.qtab[e] = make_float2((float)q, (float)dq);
            }
        }
        if (t < P.nbatch * RADT_MAXCHAN) {
            int b = t / RADT_MAXCHAN, c = t % RADT_MAXCHAN;
            double vv = (c < P.nchan) ? V.v[c] - P.vsys[b] : 0.0;
            float hi = (float)vv;
            P.ws.vcs[(size_t)(P.b0 + b) * RADT_MAXCHAN + c] = make_float2(hi, (float)(vv - (double)hi));
        }
        if (P.grid.kind != 1 && t < P.grid.n0 && P.b0 == 0) {
            // node radii of the log-spaced axis, r_i = r_min (r_max/r_min)^(i/(nr-1))
            double ri = exp2((double)t * P.grid.lg2_ratio / (double)(P.grid.n0 - 1)) / P.grid.inv_rmin;
            if (t == 0) ri = 1.0 / P.grid.inv_rmin;
            P.ws.rnode[t] = make_double2(ri, 1.0 / (ri * ri));
        }
        return;
    }
    blk -= nb_tab;
    if (blk < nb_occ && P.grid.kind == 1) {
        // 3-D occupancy: one bit per block of 4 x 4 x 4 cells, set when some node of the block's cells or of the
        // cells next to them (nodes 4I-1 .. 4I+5 per axis) stores a density that can emit (or is NaN).  One thread
        // per bit; the 32 bits of a word are the lanes of one warp.
        long long t = (long long)blk * blockDim.x + threadIdx.x;
        long long w = t >> 5;
        if (w >= (long long)P.occ_words * P.nbatch) return;
        int b = (int)(w / P.occ_words);
        int wi = (int)(w - (long long)b * P.occ_words);
        int Lw = wi % P.occ_wpr, IJ = wi / P.occ_wpr;
        int J = IJ % P.occ_nbj, I = IJ / P.occ_nbj, Lb = Lw * 32 + (threadIdx.x & 31);
        const float *dn = P.dens + (long long)(P.b0 + b) * P.batch_stride;
        bool found = false;
        if (4 * Lb < P.grid.n2 - 1) {
            int i0 = max(4 * I - 1, 0), i1 = min(4 * I + 5, P.grid.n0 - 1);
            int j0 = max(4 * J - 1, 0), j1 = min(4 * J + 5, P.grid.n1 - 1);
            int l0 = max(4 * Lb - 1, 0), l1 = min(4 * Lb + 5, P.grid.n2 - 1);
            for (int i = i0; i <= i1 && !found; ++i)
                for (int j = j0; j <= j1 && !found; ++j) {
                    const float *row = dn + ((long long)i * P.grid.n1 + j) * P.grid.n2;
                    for (int l = l0; l <= l1; ++l) found |= !(__ldg(row + l) <= P.occ_thr);
                }
        }
        unsigned word = __ballot_sync(0xffffffffu, found);
        if ((threadIdx.x & 31) == 0) P.ws.occ[(size_t)(P.b0 + b) * P.occ_words + wi] = word;
        return;
    }
    if (blk < nb_occ) {
        // Occupancy bitmap of the (r, zeta) grid for the march prefilter.  The prefilter locates a step in fp32 as
        // I = floor(u') + 1, J = floor(w') + 1 (u', w' within a small fraction of a cell of the exact index coordinates,
        // so the exact cell (i, j) has I in {i, i+1, i+2}, J likewise).  Bit J of word (I, J / 32) is therefore set when
        // some node of rows I-2 .. I+1 and columns J-2 .. J+1 -- which always include the four corners of the exact
        // cell -- stores a density that can emit (or is NaN).  occ_thr = -inf gives all ones.
        // One warp per word, lanes over the 35 node columns jw*32 - 2 .. jw*32 + 32 of each of the four rows.
        long long t = (long long)blk * blockDim.x + threadIdx.x;
        long long wq = t >> 5;
        if (wq >= (long long)P.occ_words * P.nbatch) return;
        const int ln = threadIdx.x & 31;
        int b = (int)(wq / P.occ_words);
        int w = (int)(wq - (long long)b * P.occ_words);
        int I = w / P.occ_wpr, jw = w - I * P.occ_wpr;
        const float *dn = P.dens + (long long)(P.b0 + b) * P.batch_stride;
        bool f0 = false, f1 = false;                      // column tt = ln, column tt = ln + 32 (ln < 3)
        for (int di = -2; di <= 1; ++di) {
            int ii = I + di;
            if (ii < 0 || ii >= P.grid.n0) continue;
            int j0 = jw * 32 - 2 + ln, j1 = j0 + 32;
            if (j0 >= 0 && j0 < P.grid.n1) f0 |= !(__ldg(dn + (long long)ii * P.grid.n1 + j0) <= P.occ_thr);
            if (ln < 3 && j1 < P.grid.n1) f1 |= !(__ldg(dn + (long long)ii * P.grid.n1 + j1) <= P.occ_thr);
        }
        unsigned long long m = (unsigned long long)__ballot_sync(0xffffffffu, f0) |
                               ((unsigned long long)__ballot_sync(0xffffffffu, f1) << 32);
        m |= (m >> 1) | (m >> 2) | (m >> 3);
        if (ln != 0) return;
        P.ws.occ[(size_t)(P.b0 + b) * P.occ_words + w] = (unsigned)m;
        return;
    }
    blk -= nb_occ;
    // pack SoA planes into float4 cells {dens, temp, vel, 0}; optionally zero the gradient cells.  Item by item (no 64-bit
    // division per cell), four consecutive cells per thread with 16-byte loads when the planes allow it: the pack moves 28 bytes
    // per cell (config 4: 470 MB, config 6: 352 MB per call) and ran at 2.4-3.2 TB/s with one cell per thread.
    const long long cells = P.grid.cells;
    const long long nthr = (long long)(gridDim.x - nb_rays - nb_tab - nb_occ) * blockDim.x;
    const long long tid = (long long)blk * blockDim.x + threadIdx.x;
    const bool sph_flags = P.do_pack && P.do_occ && P.grid.kind == 2;
    float tmax = 0.f;
    for (int b = 0; b < P.nbatch; ++b) {
        const long long soff = (long long)(P.b0 + b) * P.batch_stride;
        const float *dsrc = P.dens + soff, *tsrc = P.temp + soff, *vsrc = P.vel + soff;
        float4 *dst = P.ws.cells + (long long)(P.b0 + b) * cells;
        float4 *gdst = P.ws.grad + (long long)(P.b0 + b) * cells;
        unsigned *flags = P.ws.nodeflag + (size_t)(P.b0 + b) * P.grid.n0 * P.flag_wpr;
        // spherical grids: flag (i, j) when any of its phi nodes can emit (or is NaN); the flags were zeroed with the counters.
        // phi runs fastest, so the lanes of a warp normally share (i, j): one atomic per warp.
        auto flag_node = [&](long long c, bool fl) {
            const int ij = (int)(c / P.grid.n2), i = ij / P.grid.n1, j = ij - i * P.grid.n1;
            unsigned *w = flags + (size_t)i * P.flag_wpr + (j >> 5);
            const unsigned am = __activemask();
            const int leader = __ffs(am) - 1;
            if (__all_sync(am, ij == __shfl_sync(am, ij, leader))) {
                if (__any_sync(am, fl) && (int)(threadIdx.x & 31) == leader) atomicOr(w, 1u << (j & 31));
            } else if (fl) {
                atomicOr(w, 1u << (j & 31));
            }
        };
        const bool vec = !(cells & 3) && !(sph_flags && (P.grid.n2 & 3)) &&
                         (!P.do_pack || !(((size_t)dsrc | (size_t)tsrc | (size_t)vsrc) & 15));
        if (vec) {
            for (long long c4 = tid; c4 < (cells >> 2); c4 += nthr) {
                if (P.do_pack) {
                    const float4 d = __ldg(reinterpret_cast<const float4 *>(dsrc) + c4);
                    const float4 t = __ldg(reinterpret_cast<const float4 *>(tsrc) + c4);
                    const float4 v = __ldg(reinterpret_cast<const float4 *>(vsrc) + c4);
                    tmax = fmaxf(fmaxf(tmax, fmaxf(t.x, t.y)), fmaxf(t.z, t.w));
                    float4 *o = dst + 4 * c4;
                    o[0] = make_float4(d.x, t.x, v.x, 0.f); o[1] = make_float4(d.y, t.y, v.y, 0.f);
                    o[2] = make_float4(d.z, t.z, v.z, 0.f); o[3] = make_float4(d.w, t.w, v.w, 0.f);
                    if (sph_flags)      // (n2 is a multiple of 4: the four cells share (i, j))
                        flag_node(4 * c4, !(d.x <= P.occ_thr) || !(d.y <= P.occ_thr) || !(d.z <= P.occ_thr) || !(d.w <= P.occ_thr));
                }
                if (P.do_zero_grad) {
                    float4 *g = gdst + 4 * c4;
                    g[0] = g[1] = g[2] = g[3] = make_float4(0.f, 0.f, 0.f, 0.f);
                }
            }
        } else {
            for (long long c = tid; c < cells; c += nthr) {
                if (P.do_pack) {
                    const float tt = __ldg(tsrc + c), dd = __ldg(dsrc + c);
                    tmax = fmaxf(tmax, tt);
                    dst[c] = make_float4(dd, tt, __ldg(vsrc + c), 0.0f);
                    if (sph_flags) flag_node(c, !(dd <= P.occ_thr));
                }
                if (P.do_zero_grad) gdst[c] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
        }
    }
    // grid-wide maximum temperature (bounds the source function in the adjoint); counters[RADT_CNT_TMAX] holds its bits
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) tmax = fmaxf(tmax, __shfl_xor_sync(0xffffffffu, tmax, m));
    if ((threadIdx.x & 31) == 0 && tmax > 0.f) atomicMax(reinterpret_cast<int *>(P.ws.counters + RADT_CNT_TMAX), __float_as_int(tmax));
}

// Spherical occupancy words from the (i, j) node flags (second launch: needs every flag).  The prefilter locates a step in
// fp32 as I = floor(u') + 1 (radial, as on the axisymmetric grid) and C = bin of cos(theta) among n1 uniform bins over
// [pre_czlo, pre_czhi].  Bit C of word (I, C / 32) is set when some node of radial rows I-2 .. I+1 and of the theta nodes that
// a step in that bin can touch (the bin's theta range widened by one cell on both sides) is flagged.  One thread per bit.
__global__ void __launch_bounds__(256) k_occ_sph(const __grid_constant__ SetupParams P)
{
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long wq = t >> 5;
    if (wq >= (long long)P.occ_words * P.nbatch) return;
    const int ln = threadIdx.x & 31;
    const int b = (int)(wq / P.occ_words);
    const int w = (int)(wq - (long long)b * P.occ_words);
    const int I = w / P.occ_wpr, C = (w - I * P.occ_wpr) * 32 + ln;
    bool found = false;
    if (C < P.grid.n1) {
        // cos(theta) range of the bin -> theta range -> node range, one cell of margin on both sides
        const double c_lo = (double)P.grid.pre_czlo + (double)C / (double)P.grid.pre_cscale;
        const double c_hi = (double)P.grid.pre_czlo + (double)(C + 1) / (double)P.grid.pre_cscale;
        const double th_a = acos(fmin(fmax(c_hi, -1.0), 1.0)), th_b = acos(fmin(fmax(c_lo, -1.0), 1.0));      // th_a <= th_b
        const double th0 = 1.5707963267948966 - (double)P.grid.th_c0, sc = (double)P.grid.th_scale;
        const int j0 = max((int)floor((th_a - th0) * sc) - 1, 0), j1 = min((int)floor((th_b - th0) * sc) + 2, P.grid.n1 - 1);
        const unsigned *fl = P.ws.nodeflag + (size_t)(P.b0 + b) * P.grid.n0 * P.flag_wpr;
        for (int ii = max(I - 2, 0); ii <= min(I + 1, P.grid.n0 - 1) && !found; ++ii)
            for (int j = j0; j <= j1; ++j) found |= (fl[(size_t)ii * P.flag_wpr + (j >> 5)] >> (j & 31)) & 1u;
    }
    const unsigned word = __ballot_sync(0xffffffffu, found);
    if (ln == 0) P.ws.occ[(size_t)(P.b0 + b) * P.occ_words + w] = word;
}

__global__ void __launch_bounds__(256) k_unpack_grad(const float4 *__restrict__ grad, long long cells, int nbatch,
                                                     long long batch_stride, float *g_dens, float *g_temp, float *g_vel)
{
    long long total = cells * nbatch;
    long long stride = (long long)gridDim.x * blockDim.x;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += stride) {
        int b = (int)(q / cells);
        long long c = q - (long long)b * cells;
        float4 v = grad[q];
        long long dst = (long long)b * batch_stride + c;
        if (g_dens) g_dens[dst] = v.x;
        if (g_temp) g_temp[dst] = v.y;
        if (g_vel) g_vel[dst] = v.z;
    }
}

// L = 1/(2n) sum ((I - D)/sigma)^2 ; dL/dI = (I - D)/(sigma^2 n)   (chi^2 data term)
__global__ void __launch_bounds__(256) k_l2_loss_grad(const float *__restrict__ cube, const float *__restrict__ target,
                                                      float inv_s2n, double half_inv_s2n, long long n, float *dl,
                                                      double *loss)
{
    long long stride = (long long)gridDim.x * blockDim.x;
    double acc = 0.0;
    for (long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x; q < n; q += stride) {
        float r = cube[q] - target[q];
        dl[q] = r * inv_s2n;
        acc += (double)r * (double)r;
    }
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, m);
    __shared__ double part[8];
    if ((threadIdx.x & 31) == 0) part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < 8; ++w) s += part[w];
        atomicAdd(loss, s * half_inv_s2n);
    }
}

// Sum of the partial-loss slots of the fused forward (radt_march.cuh loss_report): loss = scale * sum; the slots are
// cleared for the next call.
__global__ void __launch_bounds__(RADT_LOSS_SLOTS) k_loss_finish(double *part, double scale, double *loss)
{
    double v = part[threadIdx.x];
    part[threadIdx.x] = 0.0;
#pragma unroll
    for (int m = 16; m > 0; m >>= 1) v += __shfl_xor_sync(0xffffffffu, v, m);
    __shared__ double wsum[RADT_LOSS_SLOTS / 32];
    if ((threadIdx.x & 31) == 0) wsum[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x < 32) {
        double s = wsum[threadIdx.x];
#pragma unroll
        for (int m = 16; m > 0; m >>= 1) s += __shfl_xor_sync(0xffffffffu, s, m);
        if (threadIdx.x == 0) *loss = s * scale;
    }
}

// ---------------------------------------------------------------------------------------------
// host-side launchers
// ---------------------------------------------------------------------------------------------
cudaError_t radt_launch_setup(const SetupParams &P, const LevelTable &L, const ChanTable &V, cudaStream_t st)
{
    long long nrays = (long long)P.nx * P.ny * P.nbatch;
    int nb_rays = P.do_rays ? (int)((nrays + 255) / 256) : 0;
    int need_tab = (RADT_NQ + 2) * 32;
    if (P.nbatch * RADT_MAXCHAN > need_tab) need_tab = P.nbatch * RADT_MAXCHAN;
    if (P.grid.kind != 1 && P.grid.n0 > need_tab) need_tab = P.grid.n0;
    int nb_tab = P.do_tables ? (need_tab + 255) / 256 : 0;
    long long total = P.grid.cells * P.nbatch;
    int nb_pack = 0;
    if (P.do_pack || P.do_zero_grad) {
        long long nb = (total + 255) / 256;
        nb_pack = (int)(nb < 148 * 16 ? nb : 148 * 16);
    }
    long long occ_threads = (long long)P.occ_words * P.nbatch * 32;
    int nb_occ = (P.do_occ && P.grid.kind != 2) ? (int)((occ_threads + 255) / 256) : 0;     // (spherical: radt_launch_occ_sph)
    int nb = nb_rays + nb_tab + nb_occ + nb_pack;
    if (nb == 0) return cudaSuccess;
    k_setup<<<nb, 256, 0, st>>>(P, L, V, nb_rays, nb_tab, nb_occ);
    return cudaGetLastError();
}

cudaError_t radt_launch_occ_sph(const SetupParams &P, cudaStream_t st)
{
    const long long threads = (long long)P.occ_words * P.nbatch * 32;
    k_occ_sph<<<(int)((threads + 255) / 256), 256, 0, st>>>(P);
    return cudaGetLastError();
}

cudaError_t radt_launch_unpack(const float4 *grad, long long cells, int nbatch, long long batch_stride, float *g_dens,
                               float *g_temp, float *g_vel, cudaStream_t st)
{
    long long total = cells * nbatch;
    long long nb = (total + 255) / 256;
    if (nb > 148 * 16) nb = 148 * 16;
    k_unpack_grad<<<(int)nb, 256, 0, st>>>(grad, cells, nbatch, batch_stride, g_dens, g_temp, g_vel);
    return cudaGetLastError();
}

cudaError_t radt_launch_l2(const float *cube, const float *target, double sigma, long long n, float *dl, double *loss,
                           cudaStream_t st)
{
    cudaError_t e = cudaMemsetAsync(loss, 0, sizeof(double), st);
    if (e != cudaSuccess) return e;
    double inv = 1.0 / (sigma * sigma * (double)n);
    long long nb = (n + 255) / 256;
    if (nb > 148 * 8) nb = 148 * 8;
    k_l2_loss_grad<<<(int)nb, 256, 0, st>>>(cube, target, (float)inv, 0.5 * inv, n, dl, loss);
    return cudaGetLastError();
}

cudaError_t radt_launch_loss_finish(double *part, double scale, double *loss, cudaStream_t st)
{
    k_loss_finish<<<1, RADT_LOSS_SLOTS, 0, st>>>(part, scale, loss);
    return cudaGetLastError();
}
