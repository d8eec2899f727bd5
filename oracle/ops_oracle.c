/*
 * oracle/ops_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain CPU statements of the operations SURVEY.md section 8(f) adds next to the
 * GEMM (the "NEXT" rows), under the same rules as gemm_oracle.c: only tests/,
 * __graft_entry__.smoke() and bench.py's CPU legs may load this file; it shares
 * no code with paper_2606_15991_b200/csrc.
 *
 * 1. Element-wise add (Listing 1; measured at N = 2^28 in
 *    PAPER.md:306).  The kernel of Listing 1 is
 *        let tx = x.load_like(z); let ty = y.load_like(z); z.store(tx + ty);
 *    over f32 tensors (z, x, y are Tensor<f32, ..>), one tile
 *    program per disjoint 128-element sub-tensor of z.  The
 *    paper fixes the precision (f32), so the result has a plain definition:
 *        z_i = fl32(x_i + y_i)      (one IEEE-754 binary32 addition, RNE)
 *    written here as the exact sum in binary64 rounded once to binary32.  That
 *    is the same value: binary64 carries 53 >= 2*24 + 2 significand bits, so
 *    rounding the binary64 sum of two binary32 numbers to binary32 is innocuous
 *    (the classical double-rounding condition of Figueroa).  Partitioning does
 *    not enter the value; edge tiles are masked stores, i.e.
 *    elements at index >= n are not written.
 *    Pins (tests/test_oracle_pins_ops.py): the paper's own example ones + ones
 *    over 1024 elements = 2.0 (tests/golden/listing1_add.txt), x + 0 = x,
 *    x + (-x) = +0, commutativity, ties-to-even cases at 1 + 2^-24, exact small
 *    integers, numpy's float32 add on 10^6 random pairs (library routine).
 *
 * 2. binary16 encode: binary32 -> f16 bit pattern, round to nearest even,
 *    overflow to infinity, gradual underflow.  Used only to state expected f16
 *    outputs (the GEMM's f16 output is RNE of its fp32 accumulator, DESIGN.md
 *    reading c6 applied to f16).  Pinned against numpy's astype(float16) on all
 *    finite binary32 exponent ranges, ties and 10^6 random floats; the decode is
 *    in gemm_oracle.c (dec_f16) and pinned on all 65536 patterns.
 *
 * Nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

/* z_i = fl32(x_i + y_i), i in [0, n).  Listing 1. */
void oracle_add_f32(const float *x, const float *y, float *z, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) {
        const double exact = (double)x[i] + (double)y[i]; /* exact or correctly rounded far below half an ulp32 */
        z[i] = (float)exact;                              /* the single rounding to binary32 (RNE)              */
    }
}

/* binary32 -> binary16 bits, round to nearest even. */
uint16_t oracle_f16_encode(float f)
{
    uint32_t w;
    memcpy(&w, &f, sizeof w);
    const uint16_t sign = (uint16_t)((w >> 16) & 0x8000u);
    const uint32_t a = w & 0x7fffffffu;
    if (a > 0x7f800000u) return (uint16_t)(sign | 0x7e00u);  /* NaN -> quiet NaN */
    if (a >= 0x477ff000u) return (uint16_t)(sign | 0x7c00u); /* |f| >= 65520 rounds to infinity */
    const uint32_t e = a >> 23;                              /* biased by 127 */
    if (e >= 113u) {                                         /* |f| >= 2^-14: normal binary16 */
        const uint32_t m = a & 0x7fffffu;
        uint32_t h = ((e - 112u) << 10) | (m >> 13);
        const uint32_t rem = m & 0x1fffu;                    /* the 13 dropped bits, half = 0x1000 */
        if (rem > 0x1000u || (rem == 0x1000u && (h & 1u))) ++h; /* a carry walks into the exponent */
        return (uint16_t)(sign | h);
    }
    /* subnormal binary16: multiples of 2^-24; scaling by 2^24 is exact in binary64 */
    float mag;
    memcpy(&mag, &a, sizeof mag);
    const double q = rint((double)mag * 0x1p24);             /* default rounding mode: nearest even */
    return (uint16_t)(sign | (uint16_t)q);                   /* q == 1024 is the smallest normal, 0x0400 */
}

void oracle_f16_encode_array(const float *src, uint16_t *dst, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) dst[i] = oracle_f16_encode(src[i]);
}
