// kernels.cuh — sm_100a device code of the hot path (BASELINE.json north_star subsystem (2)).
//
//   k_unpack   a1+a2 fused: raw word decode, calibration, STABLE digi/error compaction with a
//              single-pass decoupled look-back scan, modDigiStart, input-order check; TMA bulk
//              loads into a shared-memory ring, staged SoA output written by TMA bulk stores; tiles
//              handed out by an atomic ticket.
//   k_cluster  a3+a4 fused: a warp clusters a unit of up to four small modules (register packs up to 32 digis;
//              column lists + reduced edge set + atomicMin union-find on a word forest in shared memory up to 1024,
//              what does not fit the warp's region beyond some 600 digis in the global workspace), exact cluster sums and bounding boxes, cluster
//              threshold, numbering inside the module; a whole CTA (bitmap + union-find) beyond.
//   k_finalize event-wide numbering, cluster table, hit table, counters to the host.
//   k_dense    the dense path for launches whose modules are large on average: one module per CTA,
//              occupancy bitmap + popcount ranks + union-find, larger shared-memory tiers.
//   k_export   exact-size copies of requested outputs into mapped pinned host memory.
//   k_publish_digis / k_import_digis / k_occupancy   the seams of the chained modules (k_chain.cuh).
//   k_bucket / k_bucket_scan / k_unbucket_idx   words in arbitrary order: stable bucket sort by module first (A31).
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
#include "k_chain.cuh"
#include "k_bucket.cuh"
