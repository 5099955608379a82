// fft_sizes.h -- the single table of instantiated transform lengths.
// Columns: N, R1, R2, R3 (radices, R1*R2*R3 = N, R3 in {8,16}),
//          x pass: row pairs per CTA, threads;  y pass: complex columns per CTA, threads.
#pragma once

#define CANS_FFT_SIZES_A(X) \
    X(16, 2, 1, 8, 16, 32, 8, 32)    \
    X(32, 4, 1, 8, 16, 64, 8, 32)    \
    X(48, 6, 1, 8, 16, 32, 8, 32)    \
    X(64, 8, 1, 8, 16, 128, 8, 64)   \
    X(96, 12, 1, 8, 16, 128, 8, 64)   \
    X(128, 16, 1, 8, 16, 128, 8, 128)

#define CANS_FFT_SIZES_B(X) \
    X(192, 12, 1, 16, 16, 128, 8, 128)   \
    X(256, 16, 1, 16, 16, 256, 8, 128) \
    X(384, 6, 8, 8, 8, 256, 8, 256)    \
    X(512, 8, 8, 8, 8, 256, 8, 256)

#define CANS_FFT_SIZES_C(X) \
    X(768, 12, 8, 8, 4, 128, 8, 256)   \
    X(1024, 16, 8, 8, 4, 256, 4, 256)

#define CANS_FFT_SIZES_D(X) \
    X(1536, 12, 8, 16, 2, 384, 4, 256)  \
    X(2048, 16, 8, 16, 2, 256, 4, 256)

#define CANS_FFT_SIZES(X) CANS_FFT_SIZES_A(X) CANS_FFT_SIZES_B(X) CANS_FFT_SIZES_C(X) CANS_FFT_SIZES_D(X)
