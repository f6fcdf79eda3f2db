/*
 * oat_probe.h -- measurement aids of liboat.so.  NOT part of the product ABI (include/oat.h): nothing here is needed to
 * use the operators, and nothing on the operator path calls these entry points.  They serve tests (forcing the generic
 * kernel), bench.py (device time of the dominant kernel, reported diagnostics) and the micro-benchmark tables of
 * DESIGN.md section 5.3.
 */
#ifndef OAT_PROBE_H
#define OAT_PROBE_H

#include "oat.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Kernel selection for tests and measurements.  key = "project" / "backproject": variant 4 = marching kernels (default,
 * used when the geometry allows: B = 32, records indexable with 32 bits, c dt <= spacing), 0 = the generic patch kernel that
 * otherwise serves as the fall-back; "project" also takes 5 = the tile-stationary projection kernel (oat_tile.cu), which
 * holds the product tolerance.  Every selectable kernel is within 1e-4 of the oracle: "backproject" 5 (the round-2
 * tile-stationary H^T with 32-bit fixed-point accumulators, 8e-5 .. 6e-4, no overflow guard) has been removed from the
 * library and is refused; its measurement is profiles/r2_tile_bwd.md.  key = "tile_nq": transducers
 * per work item of the tile-stationary projection; "tile_tma": 0 stages the bricks with plain loads; "tile_stats": 1 collects the counters of oat_tile_stats.  key = "morton_shift": log2 of the cell size of the patch order (default 6).
 * key = "record_limit_log2": pretend record indices have that many bits (tests of the automatic fall-back).
 * Unknown key or value => OAT_ERR_INVALID. */
int oat_set_variant(oat_geometry *geom, const char *key, int variant);

/* Enumeration counters of the tile-stationary kernels, accumulated over the calls since the last reset while
 * oat_set_variant(geom, "tile_stats", 1) is in force: h_out[0] candidate rays, [1] candidates after the fp32 cull,
 * [2] rays that own at least one chunk, [3] chunks (8 samples each) marched; h_out has room for 8 values. */
int oat_tile_stats(oat_geometry *geom, unsigned long long *h_out, int reset);

/* 1 if the next oat_project (backproject = 0) / oat_backproject (backproject = 1) on this handle runs the marching
 * kernel, 0 if it runs the generic patch kernel, negative on NULL. */
int oat_uses_marching(const oat_geometry *geom, int backproject);

/* Device time (ms, CUDA events on the call's stream) of the dominant kernel of the last
 * oat_project / oat_backproject; synchronises that stream.  Negative if none was recorded. */
float oat_last_kernel_ms(oat_geometry *geom);

/* Sustained rate, in lanes per second, at which `device` retires 16-byte vector reductions (red.global.add.v4.f32)
 * that hit distinct 32-byte sectors of an L2-resident 64 MB buffer -- the path the backprojection scatter uses
 * (Alg. 6).  A diagnostic, not a roofline peak: neighbouring rays of H^T share sectors and can exceed it.
 * Allocates and frees its own scratch, synchronises the device.  Negative return on error. */
int oat_measure_red_rate(int device, double *lanes_per_s);

/* Sustained rate, in 32-byte sectors per second, at which `device` serves scattered 256-bit loads
 * (ld.global.nc.v8.f32, one distinct sector per lane) that miss L1 and hit an L2-resident 64 MB buffer -- the access
 * of the projection's marching loop (one cell record per cell run of a ray, Eq. 12 L121 / Alg. 4). */
int oat_measure_gather_rate(int device, double *sectors_per_s);

/* Parametrised forms of the two probes (tables of DESIGN.md section 5.3).
 * oat_measure_gather_rate_ex: `lanes_active` of 32 lanes load one scattered sector each, ONE load in flight per warp,
 * 8 blocks of 128 threads per SM each holding `smem_kb_per_block` KB of (unused) shared memory -- what is carved out
 * for shared memory is taken from L1.
 * oat_measure_red_rate_ex: RED.128 with an address pattern within the warp: 0 every lane its own record, 1 32 consecutive
 * records (16 sectors), 2 one record per 128-byte line, 3 lane pairs sharing a sector (regular stride), 4 four scattered lines
 * of 8 records; the sector-packing cases of a scattered accumulator (round 3): 5 every lane its own scattered sector, both
 * 16-byte halves by two back-to-back reductions of the same thread, 6 lanes l and l + 16 fill one scattered sector, 7 lanes
 * 2m and 2m + 1 fill one scattered sector.  The rate counts 16-byte reduction lanes in every pattern. */
int oat_measure_gather_rate_ex(int device, int lanes_active, int smem_kb_per_block, double *sectors_per_s);
int oat_measure_red_rate_ex(int device, int pattern, double *lanes_per_s);

#ifdef __cplusplus
}
#endif
#endif /* OAT_PROBE_H */
