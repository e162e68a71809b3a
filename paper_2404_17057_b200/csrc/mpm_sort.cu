// mpm_sort.cu -- particle re-ordering by cell key (Alg. 1 l.12) as a counting sort:
//   key_rank : key_k = linear cell index of X_k ("ptcl_to_grid"); rank_k = atomicAdd(count[key], 1)
//   scan     : exclusive prefix sum of the per-cell counts = the cell offsets / grid-to-particle connectivity
//              (the paper's steps 1(ii)-(iii))
//   permute  : every particle array is moved to offset[key] + rank in the other buffer.
// The order of particles inside one cell is the arrival order of the atomics (any order is correct, reading A17);
// results are always compared and returned by persistent id.
#include "mpm_internal.cuh"

namespace mpm {

namespace {

constexpr int kBlock = 256;
constexpr int kScanBlock = 512;
constexpr int kScanItems = 8;                       // 4096 elements per block
constexpr int kScanTile = kScanBlock * kScanItems;

__global__ void __launch_bounds__(kBlock) k_iota(int *id, long long n)
{
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k < n) id[k] = (int)k;
}

template <int DIM>
__global__ void __launch_bounds__(kBlock) k_key_rank(GridDesc gd, PArr p, int *key, int *rank, int *count, long long n)
{
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k >= n) return;
    long long cell = 0, stride = 1;
    int cc[DIM];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        double xi;
        cell_1d(p.x[a][k], gd.inv_h, gd.nc[a], cc[a], xi);
        cell += stride * cc[a];
        stride *= gd.nc[a];
    }
    if (gd.tiled) cell = tiled_key_of_cell<DIM>(gd, cc);
    key[k] = (int)cell;
    rank[k] = atomicAdd(&count[cell], 1);
}

// block-wide exclusive scan of kScanTile ints; block sums go to aux[blockIdx.x]
__global__ void __launch_bounds__(kScanBlock) k_scan_tiles(const int *in, int *data, long long n, int *aux, bool round_even)
{
    __shared__ int s_warp[kScanBlock / 32];
    const long long base = (long long)blockIdx.x * kScanTile + (long long)threadIdx.x * kScanItems;
    int v[kScanItems];
    int sum = 0;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        v[j] = (base + j < n) ? in[base + j] : 0;
        if (round_even) v[j] = (v[j] + 1) & ~1;
        sum += v[j];
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    int incl = sum;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        int t = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= o) incl += t;
    }
    if (lane == 31) s_warp[warp] = incl;
    __syncthreads();
    if (warp == 0) {
        int w = (lane < kScanBlock / 32) ? s_warp[lane] : 0;
        int wi = w;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, wi, o);
            if (lane >= o) wi += t;
        }
        if (lane < kScanBlock / 32) s_warp[lane] = wi - w;   // exclusive warp offsets
        if (lane == kScanBlock / 32 - 1) aux[blockIdx.x] = wi;
    }
    __syncthreads();
    int run = s_warp[warp] + incl - sum;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j) {
        if (base + j < n) data[base + j] = run;
        run += v[j];
    }
}

// single block: exclusive scan of aux[0..m) in place (m <= a few 10^4)
__global__ void __launch_bounds__(1024) k_scan_aux(int *aux, int m)
{
    __shared__ int s_warp[32];
    __shared__ int s_carry;
    if (threadIdx.x == 0) s_carry = 0;
    __syncthreads();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int base = 0; base < m; base += 1024) {
        const int i = base + threadIdx.x;
        const int v = (i < m) ? aux[i] : 0;
        int incl = v;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            int t = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += t;
        }
        if (lane == 31) s_warp[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            int w = s_warp[lane], wi = w;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                int t = __shfl_up_sync(0xffffffffu, wi, o);
                if (lane >= o) wi += t;
            }
            s_warp[lane] = wi - w;
        }
        __syncthreads();
        const int excl = s_carry + s_warp[warp] + incl - v;
        if (i < m) aux[i] = excl;
        __syncthreads();
        if (threadIdx.x == 1023) s_carry = excl + v;
        __syncthreads();
    }
}

__global__ void __launch_bounds__(kScanBlock) k_scan_add(int *data, long long n, const int *aux)
{
    const int add = aux[blockIdx.x];
    const long long base = (long long)blockIdx.x * kScanTile + (long long)threadIdx.x * kScanItems;
#pragma unroll
    for (int j = 0; j < kScanItems; ++j)
        if (base + j < n) data[base + j] += add;
}

template <int DIM>
__global__ void __launch_bounds__(kBlock) k_permute(PArr src, PArr dst, const int *key, const int *rank,
                                                    const int *offset, long long n)
{
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k >= n) return;
    const long long j = (long long)offset[key[k]] + rank[k];
#pragma unroll
    for (int a = 0; a < DIM; ++a) {
        dst.x[a][j] = src.x[a][k];
        dst.v[a][j] = src.v[a][k];
    }
    dst.m[j] = src.m[k];
    dst.rho[j] = src.rho[k];
    dst.e[j] = src.e[k];
    dst.q[j] = src.q[k];
    dst.id[j] = src.id[k];
}

__global__ void __launch_bounds__(kBlock) k_gather_by_id(const double *src, const int *id, double *dst, long long n)
{
    long long k = (long long)blockIdx.x * kBlock + threadIdx.x;
    if (k < n) dst[id[k]] = src[k];
}

inline unsigned grid_for(long long n, int b) { return (unsigned)((n + b - 1) / b); }

}  // namespace

void launch_iota(int *id, long long n, cudaStream_t s)
{
    if (n > 0) k_iota<<<grid_for(n, kBlock), kBlock, 0, s>>>(id, n);
}

void launch_key_rank(const GridDesc &gd, const PArr &p, int *key, int *rank, int *count, long long n, cudaStream_t s)
{
    cudaMemsetAsync(count, 0, sizeof(int) * (size_t)((gd.tiled ? gd.Nkeys : gd.Nc) + 1), s);
    if (n <= 0) return;
    if (gd.dim == 2) k_key_rank<2><<<grid_for(n, kBlock), kBlock, 0, s>>>(gd, p, key, rank, count, n);
    else k_key_rank<3><<<grid_for(n, kBlock), kBlock, 0, s>>>(gd, p, key, rank, count, n);
}

void launch_exclusive_scan_from(const int *in, int *out, long long n, int *aux, bool round_even, cudaStream_t s)
{
    if (n <= 0) return;
    const unsigned tiles = grid_for(n, kScanTile);
    k_scan_tiles<<<tiles, kScanBlock, 0, s>>>(in, out, n, aux, round_even);
    if (tiles > 1) {
        k_scan_aux<<<1, 1024, 0, s>>>(aux, (int)tiles);
        k_scan_add<<<tiles, kScanBlock, 0, s>>>(out, n, aux);
    }
}

void launch_exclusive_scan(int *data, long long n, int *aux, cudaStream_t s)
{
    launch_exclusive_scan_from(data, data, n, aux, false, s);
}

void launch_permute(const GridDesc &gd, const PArr &src, const PArr &dst, const int *key, const int *rank,
                    const int *offset, long long n, cudaStream_t s)
{
    if (n <= 0) return;
    if (gd.dim == 2) k_permute<2><<<grid_for(n, kBlock), kBlock, 0, s>>>(src, dst, key, rank, offset, n);
    else k_permute<3><<<grid_for(n, kBlock), kBlock, 0, s>>>(src, dst, key, rank, offset, n);
}

void launch_gather_by_id(const double *src, const int *id, double *dst, long long n, cudaStream_t s)
{
    if (n > 0) k_gather_by_id<<<grid_for(n, kBlock), kBlock, 0, s>>>(src, id, dst, n);
}

}  // namespace mpm
