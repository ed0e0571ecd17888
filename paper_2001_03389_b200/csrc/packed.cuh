// packed.cuh -- byte-packed device helpers shared by the uint8 kernels: PRMT wrappers, the largest / smallest byte
// of a 16-byte group (VIMNMX3.U16x2), exact per-byte masks against byte bounds, cluster / distributed-shared-memory
// wrappers.  No kernels here (a kernel lives in exactly one launch unit).
#pragma once

#include "common.cuh"

namespace rfim {

__device__ __forceinline__ uint32_t prmt_b32(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));
  return d;
}

// ---------------------------------------------------------------- cluster helpers
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_id_x() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t cluster_nid_x() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
  return r;
}
// barrier over all threads of all CTAs of the cluster; orders shared-memory accesses cluster-wide
__device__ __forceinline__ void cluster_sync_all() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t dsmem_addr(const void* local, uint32_t rank) {
  uint32_t ra;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(ra) : "r"(smem_addr(local)), "r"(rank));
  return ra;
}
__device__ __forceinline__ uint32_t dsmem_ld_u32(uint32_t addr) {
  uint32_t v;
  asm volatile("ld.shared::cluster.u32 %0, [%1];" : "=r"(v) : "r"(addr));
  return v;
}
// Exact 0xFF-per-byte mask of the bytes of w outside their column's [lo, hi]; constants per u16 lane:
// chiE/cloE for bytes 0 and 2, chiO/cloO for bytes 1 and 3 (see bytes_outside in td_u8.cuh).
__device__ __forceinline__ uint32_t bytes_outside_cols(uint32_t w, uint32_t chiE, uint32_t cloE, uint32_t chiO,
                                                       uint32_t cloO) {
  const uint32_t xe = prmt_b32(w, 0u, 0x4240u), xo = prmt_b32(w, 0u, 0x4341u);
  const uint32_t fe = (xe + chiE) | ~(xe + cloE);
  const uint32_t fo = (xo + chiO) | ~(xo + cloO);
  return prmt_b32(fe, fo, 0xFBD9u);
}

// Group summaries.  Pass T2 leaves, for every 16-byte group of the row, its largest and its smallest byte
// (two byte arrays gmax[], gmin[]).  A cut with kept interval [lo, hi] touches a group iff max > hi or
// min < lo, so the threshold sweeps read two bytes per group instead of sixteen.  For a 32-bit word w the u16 lanes of w and of w << 8 carry every
// byte once as the HIGH byte of a lane (the low byte is junk that cannot change the order of the high
// bytes), so VIMNMX3.U16x2 over {x, y, z, w, x<<8, y<<8, z<<8, w<<8} gives the lane with the largest / smallest byte.
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t d;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(d) : "r"(a), "r"(b), "r"(sel));   // selector bit 3 = replicate sign
  return d;
}
__device__ __forceinline__ uint32_t group_summary(const uint4& w) {
  const uint32_t x0 = w.x << 8, x1 = w.y << 8, x2 = w.z << 8, x3 = w.w << 8;
  uint32_t mx = __vimax3_u16x2(w.x, w.y, w.z), mn = __vimin3_u16x2(w.x, w.y, w.z);
  mx = __vimax3_u16x2(mx, w.w, x0); mn = __vimin3_u16x2(mn, w.w, x0);
  mx = __vimax3_u16x2(mx, x1, x2);  mn = __vimin3_u16x2(mn, x1, x2);
  mx = __vmaxu2(mx, x3);            mn = __vminu2(mn, x3);
  mx = __vmaxu2(mx, prmt(mx, mx, 0x1032u));                   // both lanes: the lane with the largest high byte
  mn = __vminu2(mn, prmt(mn, mn, 0x1032u));
  return prmt(mx, mn, 0x4415u);                               // byte 1 = max byte, byte 0 = min byte
}
// the same for the four words of a group held by four neighbouring lanes (fix path): summary in every lane
__device__ __forceinline__ uint32_t quad_summary(uint32_t w, uint32_t mask) {
  const uint32_t x = w << 8;
  uint32_t mx = __vmaxu2(w, x), mn = __vminu2(w, x);
  mx = __vmaxu2(mx, __shfl_xor_sync(mask, mx, 1)); mn = __vminu2(mn, __shfl_xor_sync(mask, mn, 1));
  mx = __vmaxu2(mx, __shfl_xor_sync(mask, mx, 2)); mn = __vminu2(mn, __shfl_xor_sync(mask, mn, 2));
  mx = __vmaxu2(mx, prmt(mx, mx, 0x1032u));
  mn = __vminu2(mn, prmt(mn, mn, 0x1032u));
  return prmt(mx, mn, 0x4415u);
}
// byte masks (0xFF per byte) of the bytes of w that are > hi / < lo; cab2 = 0x7fff - hi, cbe2 = 0x7fff + lo in
// both u16 halves: lane + cab2 has bit 15 set iff byte > hi, cbe2 - lane has bit 15 set iff byte < lo
__device__ __forceinline__ uint32_t bytes_above(uint32_t w, uint32_t cab2) {
  return prmt(prmt(w, 0u, 0x4240u) + cab2, prmt(w, 0u, 0x4341u) + cab2, 0xFBD9u);
}
__device__ __forceinline__ uint32_t bytes_below(uint32_t w, uint32_t cbe2) {
  return prmt(cbe2 - prmt(w, 0u, 0x4240u), cbe2 - prmt(w, 0u, 0x4341u), 0xFBD9u);
}

// Exact mask (0xFF per byte) of the bytes of w outside [lo, hi], 9 instructions: the bytes are spread
// over two words of u16 lanes; lane + (0x7FFF - hi) sets bit 15 iff byte > hi, lane + (0x8000 - lo)
// sets bit 15 iff byte >= lo; PRMT's sign-replicate mode turns the four bit-15 flags into a byte mask.
// chi2 / clo2 hold those constants in both halves.  With lo = 1, hi = 0 every byte is marked.
__device__ __forceinline__ uint32_t bytes_outside(uint32_t w, uint32_t chi2, uint32_t clo2) {
  const uint32_t xe = prmt(w, 0u, 0x4240u), xo = prmt(w, 0u, 0x4341u);
  const uint32_t fe = (xe + chi2) | ~(xe + clo2);
  const uint32_t fo = (xo + chi2) | ~(xo + clo2);
  return prmt(fe, fo, 0xFBD9u);
}

}  // namespace rfim
