/* include/vr_measure.h — measurement and test aids of libvr_b200.so, kept apart from the product boundary (include/vr.h,
 * SURVEY.md section 8(b)).  bench.py and tests/ use them; a viewer does not need them.  Same conventions as vr.h:
 * d_ pointers are DEVICE memory, everything else HOST; every call returns a vr_status.  These calls synchronise and
 * may allocate scratch memory on the device.
 */
#ifndef VR_MEASURE_H
#define VR_MEASURE_H

#include "vr.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement aids (not on the product path):
 * vr_measure: renders the frame with the instrumented build of the caster and returns, in HOST
 *     counters, the lattice samples visited (every sample of O4 up to early termination: the oracle's
 *     count) and the number of distinct 32-byte sectors of the tiled cube that the evaluated samples'
 *     2x2x2 footprints touched (algorithmic HBM bytes of the cube = 32 * that).
 *     Synchronises.  Either output may be NULL.                                                  */
vr_status vr_measure(vr_volume* vol, const vr_camera* cam, int W, int H, float step_voxels, int mode,
                     float ert_alpha, long long* h_samples, long long* h_sectors);
/* vr_measure_units: the full set of counters of the instrumented caster (which takes the same skip and termination
 *     decisions as the product caster).  h_samples[0] = lattice samples visited (= vr_measure's, the oracle's
 *     count), h_samples[1] = samples evaluated (visited minus those empty-space skipping passed over).
 *     h_units[0..2] = distinct 32-byte sectors (= vr_measure's), 64-byte sector pairs and 128-byte lines of the
 *     tiled cube that the EVALUATED samples' footprints touched — what a memory system fetching 32, 64 or 128
 *     bytes per miss has to move; h_units[3] = distinct 32-byte sectors of the occupancy mask that were read.
 *     Either array may be NULL.                                                                                 */
vr_status vr_measure_units(vr_volume* vol, const vr_camera* cam, int W, int H, float step_voxels, int mode,
                           float ert_alpha, long long h_samples[2], long long h_units[4]);
/* Device time, in ms, of the cast kernel and of the composite kernel of the most recent vr_render /
 *     vr_render_to_host on this volume (CUDA events recorded on the volume's stream around each
 *     launch; composite is 0 when a single brick wrote the frame directly).  Waits for that frame. */
vr_status vr_get_stage_ms(vr_volume* vol, float* h_cast_ms, float* h_composite_ms);
/* Device time of the re-layout kernel of vr_create_volume, in ms, and the bytes it allocated.  */
vr_status vr_volume_info(const vr_volume* vol, float* h_relayout_ms, long long* h_tiled_bytes);
/* Inverse of the re-layout: gathers the tiled copy back into d_linear[nz][ny][nx] (round-trip test). */
vr_status vr_export_linear(vr_volume* vol, float* d_linear);

#ifdef __cplusplus
}
#endif
#endif /* VR_MEASURE_H */
