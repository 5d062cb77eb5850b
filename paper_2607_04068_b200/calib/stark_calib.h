/*
 * stark_calib.h -- measurement aids of `bench.py --calibrate` ("launch-floor
 * calibration").  NOT part of the product ABI (include/stark.h): built into its own
 * libstark_calib.so, loaded only by paper_2607_04068_b200/calib/__init__.py.
 *
 * stark_calib_empty: launches an empty kernel -- the launch floor.
 * stark_calib_stream_read: a plain grid-stride 16-byte read of `bytes` bytes of device memory `src`
 * (148*8 CTAs of 256 threads, 4 loads in flight per thread) -- what a trivial HBM-bound kernel of that
 * size achieves, launch and ramp included; `sink` must point to 4 writable device bytes (never written
 * unless the data XORs to a magic value).  `stream` is a cudaStream_t.
 * Return: 0, -1 (null pointer / bytes < 16) or -4 (a CUDA call failed).
 */
#ifndef STARK_CALIB_H_
#define STARK_CALIB_H_
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif
int stark_calib_empty(void* stream);
int stark_calib_stream_read(const void* src, size_t bytes, void* sink, void* stream);
#ifdef __cplusplus
}
#endif
#endif
