// fast_configs.hpp -- the line lengths that have a register-resident Stockham instantiation, with their
// radices (first radix a power of two that divides the largest one; radices 5 and 6 go last) and tile shapes.
#pragma once

// x direction: complex line length N = nx / 2 -> (N, R0, R1, R2)
#define FSEI_X_CONFIGS(X) \
    X(16, 4, 4, 1) X(32, 8, 4, 1) X(64, 8, 8, 1) X(128, 8, 16, 1) X(256, 16, 16, 1) X(512, 8, 8, 8) X(1024, 16, 8, 8) \
    X(48, 8, 6, 1) X(96, 16, 6, 1) X(192, 8, 4, 6) X(384, 8, 8, 6) \
    X(80, 16, 5, 1) X(160, 8, 4, 5) X(320, 8, 8, 5) X(640, 16, 8, 5) \
    X(240, 8, 6, 5) X(288, 8, 6, 6) X(480, 16, 6, 5) X(576, 16, 6, 6)

// y direction: column length N = ny -> (N, R0, R1, R2, CY); CY adjacent slots (CY * 16 contiguous bytes) per tile row
#define FSEI_Y_CONFIGS(X) \
    X(16, 4, 4, 1, 8) X(32, 8, 4, 1, 8) X(64, 8, 8, 1, 8) X(128, 8, 16, 1, 8) X(256, 16, 16, 1, 8) X(512, 8, 8, 8, 4) \
    X(1024, 16, 8, 8, 4) X(48, 8, 6, 1, 8) X(96, 16, 6, 1, 8) X(192, 8, 4, 6, 8) X(384, 8, 8, 6, 4) X(768, 16, 8, 6, 4) \
    X(80, 16, 5, 1, 8) X(160, 8, 4, 5, 8) X(320, 8, 8, 5, 8) X(640, 16, 8, 5, 4) X(1280, 16, 16, 5, 4) \
    X(240, 8, 6, 5, 8) X(288, 8, 6, 6, 8) X(480, 16, 6, 5, 4) X(576, 16, 6, 6, 4) X(960, 16, 6, 10, 4) X(1152, 16, 6, 12, 4)

// Fused path (blocked spectrum, z-marching y kernels of yzfused.cuh): slots per tile, and the lengths it is
// instantiated for -- the large grids, where one CTA per x-slot tile fills the GPU.
#define FSEI_CB 2
// x direction, blocked stores / loads: (N, R0, R1, R2) -- same radices as FSEI_X_CONFIGS
// (the short lengths are never chosen by the plan; FSEI_PATH=fused reaches them so that tests can run the fused kernels
// on grids the oracle and the host harness finish in seconds)
#define FSEI_XB_CONFIGS(X) X(256, 16, 16, 1) X(512, 8, 8, 8) X(1024, 16, 8, 8) X(384, 8, 8, 6) X(320, 8, 8, 5) X(640, 16, 8, 5) \
    X(288, 8, 6, 6) X(480, 16, 6, 5) X(576, 16, 6, 6) X(16, 4, 4, 1) X(32, 8, 4, 1) X(48, 8, 6, 1) X(160, 8, 4, 5)
// y direction: (N, R0, R1, R2) -- same radices as FSEI_Y_CONFIGS
#define FSEI_YZ_CONFIGS(X) X(384, 8, 8, 6) X(512, 8, 8, 8) X(768, 16, 8, 6) X(1024, 16, 8, 8) X(640, 16, 8, 5) X(1280, 16, 16, 5) \
    X(480, 16, 6, 5) X(576, 16, 6, 6) X(960, 16, 6, 10) X(1152, 16, 6, 12) X(16, 4, 4, 1) X(32, 8, 4, 1) X(48, 8, 6, 1) X(160, 8, 4, 5)
