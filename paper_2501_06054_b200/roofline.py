"""ALU roofline of the trace kernel.

The path moves almost no HBM bytes (<= 0.04 B per neutron) and has no dense contraction: it is bound
by instruction issue on the plain ALUs.  One SM sub-partition (SMSP; 4 per SM, 148 SMs) issues at most
one warp instruction per clock; FP64 instructions additionally occupy the 16-lane FP64 pipe for 2
clocks and MUFU/conversion instructions the 4-lane XU pipe for 8 clocks.  The roofline of a config is
therefore the largest of three per-neutron costs, in SMSP-clocks per 32 neutrons:

    issue = all algorithmic thread-instructions          (1 clock per warp instruction)
    fp64  = 2 x FP64 thread-instructions
    xu    = 8 x MUFU/conversion thread-instructions
    imul  = 4 x 32x32->64-bit integer multiplies         (Philox: 20 per block, the heavy FMA pipe)

The clocks per warp instruction are MEASURED on the B200 with csrc/microbench.cu (profiles/r1_microbench.md):
FFMA 1.04, IMAD 2.02, IMAD.WIDE 4.05 inside Philox (a whole Philox4x32-10 block: 81 clocks), LOP3 2.03,
DFMA 2.03, MUFU 8.05.

The per-unit instruction counts below are ALGORITHMIC: the arithmetic that the method, in the
formulation this library uses, needs on this ISA (a fp64 division = 1 MUFU.RCP64H + 9 DFMA-class,
a fp64 sqrt = 1 MUFU.RSQ64H + 9, fp64 sincos = 62, Philox4x32-10 = 40 integer instructions, ...),
counted per unit of work: every launched neutron (stage A), every slit-1 survivor (stage B0: Philox
block 1 and the certain-miss test), every survivor whose geometry is evaluated (stage B), every
detected neutron (stage-C prologue) and every quadrature node evaluation.  The per-node counts are the
arithmetic instructions (FFMA/FMUL/FADD/MUFU/select) of the shipped loop bodies, read from the SASS of
this build (cuobjdump): table loads, loop control, register moves, queue handling, work fetching and
atomics are NOT in them, so the fraction cannot exceed the kernel's issue-slot utilisation.  The unit
fractions (survivors, evaluated geometries, detected per launched neutron) are the counters of the
timed run itself.
"""
from __future__ import annotations

N_SM = 148
SMSP_PER_SM = 4
SM_MAX_MHZ = 1965.0

# thread-instructions per unit: (issue_total, fp64, xu, wide integer multiplies)
STAGE_A = (46, 0, 0, 19)        # Philox block 0 (40; the last round needs one of its two products) + id/compare (6)
STAGE_B0 = (40 + 12, 12, 0, 20) # Philox block 1 (40) + two uniforms, q, lambda, q*lambda test in fp64 (12)
# Philox block 0 again (40) + 8 uniforms (3 fp64 each) + ~125 fp64 add/mul/compare + 8 div (10) + 3 sqrt (10)
# + sincos (62) + floor/convert (6 xu-class conversions)
STAGE_B = (40 + 24 + 125 + 80 + 30 + 62 + 12, 24 + 125 + 72 + 27 + 62, 11 + 6, 20)

# per detected neutron: prologue (|Q|, projections, weight product, 3 atomics) and per node evaluation
MODEL_COST = {
    # name: (prologue(issue, fp64, xu), per_node(issue, fp64, xu))
    "sphere_fp64": ((40, 30, 2, 0), (110, 100, 2, 0)),
    "sphere_fp32": ((40, 30, 4, 0), (32, 0, 1, 0)),
    "sphere_py_fp32": ((40 + 60, 30, 5, 0), (32, 0, 1, 0)),
    "sphere_py_fp64": ((40 + 160, 30 + 150, 4, 0), (110, 100, 2, 0)),
    "cylinder_quad_fp32": ((60, 40, 4, 0), (27, 0, 1, 0)),
    "cs_triaxial_iso_fp32": ((40 + 40 + 90, 120, 6, 20), (33, 0, 2, 0)),
    "cylinder_iso_fp64": ((40 + 40 + 200 + 320, 520, 8, 20), (0, 0, 0, 0)),
    # per-event sizes: Philox blocks 2 and 3, two Box-Muller normals (log, sqrt, cos in fp64), three sincospi,
    # sin, j1, the weight
    "cylinder_event_fp64": ((40 + 80 + 260 + 200 + 320, 780, 12, 40), (0, 0, 0, 0)),
    # barbell, per event: the cylinder term and the prologue of the per-event path, then 64 slice evaluations
    # (square root, fp64 J1, fp64 cos, ~15 multiply-adds: ~95 instructions of which ~30 FP64, from the ncu
    # instruction and pipe counts of the n2 workload: 491 thread instructions and 143 FP64 per launched neutron)
    "barbell_event_fp64": ((40 + 80 + 260 + 200 + 320, 780, 12, 40), (95, 30, 2, 0)),
}

# DRAM traffic of one trace-kernel launch, dram__bytes_read.sum + dram__bytes_write.sum of the
# `ncu --set full` captures summarised in profiles/r1_ncu_c<k>.md (bytes per launch; c4: the first of its
# two launches, the 512 sphere experiments).  The algorithmic traffic is the histograms only.
NCU_DRAM_BYTES = {
    "c0_sphere_fp64": 445_696,
    "c1_polysphere_py": 1_626_880,
    "c2_oriented_cylinder": 1_683_712,
    "c3_coreshell_triaxial": 6_359_040,
    "c4_batch": 351_287_296,
}


def smsp_clocks_per_neutron(frac_survive: float, frac_detect: float, model_key: str, nodes: int,
                            frac_geometry: float | None = None):
    """Algorithmic SMSP-clocks per launched neutron (per lane: divide by 32 for per-warp) for each
    resource; returns dict(issue=, fp64=, xu=, imul=)."""
    pro, node = MODEL_COST[model_key]
    if frac_geometry is None:
        frac_geometry = frac_survive      # no classifier: every survivor's geometry is evaluated
    tot = [0.0, 0.0, 0.0, 0.0]
    for i in range(4):
        tot[i] = (STAGE_A[i] + frac_survive * STAGE_B0[i] + frac_geometry * STAGE_B[i]
                  + frac_detect * (pro[i] + nodes * node[i]))
    return dict(issue=tot[0], fp64=2.0 * tot[1], xu=8.0 * tot[2], imul=4.0 * tot[3])


def roofline(neutrons_per_s: float, frac_survive: float, frac_detect: float, model_key: str, nodes: int,
             sm_mhz: float = SM_MAX_MHZ, workload: str | None = None, frac_geometry: float | None = None):
    """Roofline record for bench.py.  `achieved` and `peak` are in G thread-instructions/s on the
    binding resource (issue slots x 32 lanes: 148 SM x 4 SMSP x 32 lanes x clock)."""
    c = smsp_clocks_per_neutron(frac_survive, frac_detect, model_key, nodes, frac_geometry)
    pipe = max(c, key=c.get)
    peak_lane_clocks = N_SM * SMSP_PER_SM * 32 * sm_mhz * 1e6      # lane-clocks per second
    achieved = neutrons_per_s * c[pipe]
    # the same path without the classifier shortcut (every survivor's geometry evaluated): what a plain
    # implementation of DESIGN.md section 3 would have to issue for this throughput
    plain = smsp_clocks_per_neutron(frac_survive, frac_detect, model_key, nodes, frac_survive)
    return {
        "bound": "alu", "pipe": pipe,
        "achieved": achieved / 1e9, "peak": peak_lane_clocks / 1e9, "unit": "G lane-clocks/s",
        "frac": achieved / peak_lane_clocks,
        "frac_plain_algorithm": neutrons_per_s * max(plain.values()) / peak_lane_clocks,
        "alg_clocks_per_neutron": {k: round(v, 2) for k, v in c.items()},
        "peak_source": f"derived: {N_SM} SM x {SMSP_PER_SM} SMSP x 32 lanes x {sm_mhz:.0f} MHz (DESIGN.md s.7)",
        "traffic": NCU_DRAM_BYTES.get(workload),
    }
