// kernels.cuh — sm_100a device code of the hot path (BASELINE.json north_star subsystem (2)).
//
//   k_unpack   a1+a2 fused: raw word decode, calibration, STABLE digi/error compaction with a
//              single-pass decoupled look-back scan, modDigiStart, input-order check; TMA bulk
//              loads into a shared-memory ring, staged SoA output written by TMA bulk stores.
//   k_cluster  a3+a4 fused: per-module 8-connected components (one warp per pack of small modules:
//              all in registers; per module of 33..256 digis: hash look-up + label equivalence in
//              shared memory; CTA per large module: bitmap + rank look-up + min-index union-find),
//              exact cluster sums, cluster threshold, per-module numbering.
//   k_dense    the large-module path of k_cluster as a kernel of its own (larger shared-memory tiers), used
//              by launches whose modules are large on average.
//   k_finalize event-wide dense cluster numbering, cluster SoA, modClusStart, counters to the host.
//   k_export   exact-size copies of requested outputs into mapped pinned host memory.
//
// Kernels are batch-capable: a launch processes nEv independent events described by EvDesc
// records (one Run-3-like event is ~1000x too small to fill a B200).  The single-event path
// passes its descriptor as a __grid_constant__ kernel parameter (no descriptor upload).
//
// The paper describes no kernel; its only constraint on device code is "no
// assert() in kernel code" (L88): errors are reported through a status word, never trapped.
// Definitions of every quantity: DESIGN.md, readings A1-A14.  Shares nothing with oracle/.
#pragma once
#include "common.cuh"
#include "k_unpack.cuh"
#include "k_cluster.cuh"
#include "k_finalize.cuh"
