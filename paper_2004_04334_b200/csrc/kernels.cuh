// kernels.cuh — sm_100a device code of the hot path (BASELINE.json north_star subsystem (2)).
//
//   k_unpack   a1+a2 fused: raw word decode, calibration, STABLE digi/error compaction with a
//              single-pass decoupled look-back scan, modDigiStart, input-order check; TMA bulk
//              loads into a shared-memory ring, staged SoA output written by TMA bulk stores; tiles
//              handed out by an atomic ticket.
//   k_cluster  a3+a4+hits fused, one CTA per unit of consecutive modules, one thread per digi:
//              shared-memory hash + min-index union-find, exact cluster sums by 32-bit limb
//              reductions, cluster threshold, EVENT-WIDE numbering by a look-back over the units,
//              cluster and hit tables, counters to the host.  One pass, nothing re-read.
//   k_dense    the same for launches whose modules are large on average: one module per CTA,
//              occupancy bitmap + popcount ranks + union-find, larger shared-memory tiers.
//   k_export   exact-size copies of requested outputs into mapped pinned host memory.
//   k_publish_digis / k_import_digis / k_occupancy   the seams of the chained modules (k_chain.cuh).
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
