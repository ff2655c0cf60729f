/* cos(2 pi k / 48), k = 0..12, correctly rounded binary64 literals -- do not edit.
 * How they were made: a one-off script evaluated cos by its Taylor series with Python's decimal module at 60 digits
 * (pi from Machin's formula) and rounded once to binary64; tests/test_host_logic.py checks the table against
 * math.cos to 1 ulp.  Every in-register butterfly constant of the FFT codelets (radices 2 ... 16, all divisors of 48)
 * comes from this table; the CPU oracle does not use it (it calls cosl / sinl). */
#pragma once
#define TDH_COS48_TABLE { \
    1.0, /* k=0 */ \
    0.9914448613738104, /* k=1 */ \
    0.9659258262890683, /* k=2 */ \
    0.9238795325112867, /* k=3 */ \
    0.8660254037844386, /* k=4 */ \
    0.7933533402912352, /* k=5 */ \
    0.7071067811865476, /* k=6 */ \
    0.6087614290087207, /* k=7 */ \
    0.5, /* k=8 */ \
    0.3826834323650898, /* k=9 */ \
    0.25881904510252074, /* k=10 */ \
    0.1305261922200516, /* k=11 */ \
    0.0 /* k=12 */ \
}
