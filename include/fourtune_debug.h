/* fourtune_debug.h -- test / bench hooks of libfourtune.so.  NOT part of the product interface
 * (include/fourtune.h): process-global switches that force a kernel variant so that the parity tests
 * can cover every variant on every shape.  Not thread-safe; set them while no call is in flight. */
#ifndef FOURTUNE_DEBUG_H_
#define FOURTUNE_DEBUG_H_

#ifdef __cplusplus
extern "C" {
#endif

/* GEMM variant: 0 = default (the library picks the CTA-pair kernel and its tile width per shape);
 * 128, 192, 256 = the 1-CTA kernel with that N tile (kept as a cross-check of the pair kernel);
 * 1000 + bn = the CTA-pair kernel with tile width bn (bn = 256: scale columns overlaid on the draining
 * accumulator; bn = 224 / 240: scale columns of their own; falls back to 256 if the weight operand carries no
 * scales cut to that width). */
int ft_debug_set_gemm_tile_n(int bn);
/* quantizer route: 0 = default (single-pass amax + quantize when the tensor fits the SMs' shared memory),
 * 1 = always the two-pass path (k_amax, then the streaming quantize kernel) */
int ft_debug_set_quantize_mode(int mode);

#ifdef __cplusplus
}
#endif
#endif /* FOURTUNE_DEBUG_H_ */
