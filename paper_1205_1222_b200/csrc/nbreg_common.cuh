// nbreg_common.cuh -- shared definitions of the CUDA path (no arithmetic of the method lives here).
//
// Packed predicted j-records ("Jparticle" of Listing B1, redesigned): the predictor
// writes, and the force kernel streams through shared memory, one 80-byte record per PAIR of consecutive
// j-particles (j0 = 2p, j1 = 2p + 1), laid out so that each 16-byte quarter feeds one packed f32x2
// instruction operand pair directly:
//     q0 = { xh0, xh1, yh0, yh1 }     position high words   (xh = fl32(x_p))
//     q1 = { zh0, zh1, m0,  m1  }
//     q2 = { vx0, vx1, vy0, vy1 }     velocity, fl32
//     q3 = { vz0, vz1, xl0, xl1 }     position low words    (xl = fl32(x_p - xh): "two-float")
//     q4 = { yl0, yl1, zl0, zl1 }
// The low words sit at the end of the record: the common (far-pair) path of the force kernel never loads them.
// = 40 B per j.  A second, PARTICLE-major copy serves kernels that gather single particles by index (the irregular
// force, irregular.cuh): three float4 per particle, { xh, yh, zh, m } { xl, yl, zl, vx } { vy, vz, 0, 0 } = 48 B in
// two 32-byte sectors, against three or four sectors and five accesses for a particle's half of a pair record.
// The pair array is padded with massless dummies parked far away up to a multiple of kJPad.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace nbreg {

constexpr int kQuadsPerPair = 5;       // float4 per packed j-pair
constexpr int kGatherQuads = 3;        // float4 per particle of the particle-major copy (below)
constexpr int kBytesPerJ = 40;         // packed bytes per j-particle
constexpr int kJPad = 256;             // packed array length is a multiple of this (largest j-tile)
constexpr float kFarAway = 1.0e18f;    // coordinate of the massless padding particles
constexpr int kMaxChunks = 4096;       // most j-chunks a row block is split into
constexpr int kMaxNbrCap = 8192;       // nbr_cap limit: the gather kernel stages 4 rows of cap entries in shared memory

__host__ __device__ inline int64_t round_up(int64_t a, int64_t b) { return (a + b - 1) / b * b; }

// Programmatic dependent launch (sm_90+): the kernels of one call are launched with the programmatic-stream-
// serialization attribute, so that a kernel's launch latency overlaps the tail of the kernel before it.  Every such
// kernel calls pdl_wait() before it touches global memory (it returns once ALL earlier kernels of the stream have
// completed and their writes are visible; a no-op for a kernel launched the ordinary way).  pdl_trigger() lets the next
// kernel of the stream be scheduled once every CTA of this one has got that far (or has exited).  It sits LATE in the
// kernels, after their main loop: CTAs of the next kernel that are resident while they wait take issue slots from the
// CTAs still computing (measured: triggering at the start of force_kernel cost a 512-row call at N = 65536 14 %).
#ifndef NBREG_PDL_TRIGGER
#define NBREG_PDL_TRIGGER 1
#endif
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() {
#if NBREG_PDL_TRIGGER
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
}

}  // namespace nbreg
