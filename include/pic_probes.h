/*
 * pic_probes.h -- C ABI of libpic_probes.so: measurement tools for bench.py and
 * DESIGN.md section 5, NOT part of the simulation library (include/pic.h).
 * Return codes are pic.h's: 0 = PIC_OK, -1 = PIC_EINVAL, -2 = PIC_ENOMEM,
 * -3 = PIC_ECUDA.
 */
#ifndef PIC_B200_PROBES_H
#define PIC_B200_PROBES_H

#ifdef __cplusplus
extern "C" {
#endif

/*
 * Micro-probes of the machine rates the rooflines are quoted against
 * ("Builder must measure first: fp64 FMA peak ...,
 * shared-memory LDS.64 wavefront rate with 1/2/4 distinct addresses per warp
 * ..., global fp64 red.add rate at L2").  Not part of a simulation: no ctx;
 * they run on the current CUDA device and the default stream, allocate a few
 * MB of device scratch themselves (cudaMalloc) and free it before returning --
 * which is why they live in a library of their own, libpic_probes.so, and not
 * in libpic_b200.so: the product library never allocates device memory.  All pointers are HOST pointers.
 * Return PIC_OK, PIC_EINVAL (bad argument), PIC_ENOMEM or PIC_ECUDA.
 *
 * pic_probe_dfma: clocks per warp-wide DFMA per SM with `warps_per_sm` warps
 *   of 8 independent dependent chains each (one block per SM, clock64).
 * pic_probe_dmma: clocks per warp-wide DMMA m8n8k4 (256 fp64 FMA) per SM, 8
 *   independent accumulator fragments per warp.
 * pic_probe_lds: clocks per warp-wide LDS.64 (vec_bytes 8) or LDS.128 (16) per
 *   SM.  Lane l of every warp reads the fp64 word lane_word[l] (32 ints; even
 *   for LDS.128) of a 6,144-word shared array, eight independent loads per
 *   loop trip, load k displaced by k*plane_words words; lanes whose bit in
 *   active_mask is 0 leave before the loop.
 * pic_probe_red: lane-level red.global.add.f64 per second over the whole GPU
 *   (8 blocks of 256 threads per SM, CUDA events) into `footprint_doubles`
 *   doubles.  pattern 0: a warp adds to 32 consecutive doubles; 1: one 32-byte
 *   sector per lane; 2: one 128-byte line per lane; 3: all lanes one double;
 *   4: 8 unrelated places x 4 planes `plane_doubles` apart (an unmerged
 *   per-cell accumulator flush); 5: 8 unrelated places x 4 consecutive doubles.
 */
int pic_probe_dfma(int warps_per_sm, int iters, double* clk_per_warp_instr);
int pic_probe_dmma(int warps_per_sm, int iters, double* clk_per_warp_instr);
int pic_probe_lds(int vec_bytes, const int* lane_word, unsigned int active_mask, int plane_words,
                  int warps_per_sm, int iters, double* clk_per_warp_instr);
int pic_probe_red(int pattern, long long footprint_doubles, long long plane_doubles,
                  int reds_per_thread, double* lane_reds_per_s);

#ifdef __cplusplus
}
#endif
#endif /* PIC_B200_PROBES_H */
