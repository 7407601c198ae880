"""ALU roofline of the trace kernels.

The path moves almost no HBM bytes (<= 0.04 B per neutron) and has no dense contraction: it is bound by the
integer, FP64, FP32 and special-function units of the SM sub-partitions (SMSP; 4 per SM, 148 SMs).  A config's
bound is the largest of five per-neutron costs, in SMSP clocks per lane (x 32 = per warp row):

    issue = c_ffma  x all algorithmic thread-instructions            (the issue port; FFMA runs at that rate)
    imul  = c_wide  x 32x32->64 multiplies + c_imad x 32-bit multiplies   (the integer multiplier, "FMA heavy" pipe)
    int   = c_lop3  x logic-pipe instructions + c_wide_int x 32x32->64 multiplies
    fp64  = c_dfma  x FP64 instructions
    xu    = c_mufu  x MUFU / POPC / conversion instructions
    fma   = (imul + c_ffma2 x FP32 operations) / 2               (the two FMA pipes, heavy and lite, 16 lanes each)

An FP32 operation occupies one of the two FMA pipes for two clocks, a packed one (FFMA2 / FMUL2 / FADD2: two
operations per lane in one instruction; c_ffma2, measured by the microbenchmark: 2.02 clocks per warp instruction)
both of them; the integer
multiplies run on the heavy pipe only.  The packed node loops of c2 and c3 count one ISSUE slot per packed
instruction and two FP32 operations: they are bound by `fma`, no longer by `issue`.

The clocks per warp instruction (c_*) are MEASURED on the box by csrc/microbench.cu, which bench.py runs before
timing anything (`rates` below holds the figures of profiles/r2_microbench.md as a fallback only):
FFMA 1.04, IMAD 2.02, LOP3 2.02, DFMA 2.03, MUFU 8.04; a 32x32->64 multiply occupies the multiplier for 4.05
clocks AND keeps the logic pipe from issuing for 2.05 of them: a stream of one multiply plus n LOP3 takes
2.02 n + 2.05 clocks for every n >= 1 (measured 4.14, 6.10, 8.08, 10.07 for n = 1..4), so a Philox4x32-10 block
(20 multiplies, 20 LOP3) costs 81 clocks on both pipes at once and every further logic instruction of stage A
adds two full clocks.  `int` is that law.  It is checked against the kernel's own arithmetic: the stage-A core
(words 0, 1 of Philox block 0 plus the window test, microbench `stage_a_core_row`) measures 76.1 clocks per row
where the law gives 2.02 x 19.7 + 2.05 x 16 = 72.6 and the multiplier alone 66.

The per-unit instruction counts are ALGORITHMIC: the arithmetic (multiplies, logic/compare/select, FP64, FP32,
MUFU/POPC/conversions) of the shipped code of each stage, counted from the executed SASS of this build with the
ncu source page (profiles/r2_instruction_counts.md): loads, stores, atomics, address arithmetic, moves, branches,
barriers, queue handling and work fetching are NOT in them, nor are two things the kernels do for their own
convenience -- the second draw of Philox block 0 in stage B and the certain-miss classifier of stage B0.  The
fraction therefore cannot exceed the kernel's issue-slot utilisation.  The unit frequencies (survivors,
evaluated geometries, detected per launched neutron) are the counters of the timed run itself.
"""
from __future__ import annotations

N_SM = 148
SMSP_PER_SM = 4
SM_MAX_MHZ = 1965.0

# fallback rates: profiles/r2_microbench.md (B200, 1965 MHz); bench.py replaces them with the live run
RATES = dict(ffma=1.036, ffma2=2.02, imad=2.020, imad_wide=4.05, lop3=2.024, dfma=2.029, mufu=8.04, wide_int=2.05,
             philox_block=81.0, stage_a_core_row=76.1, source="profiles/r2_microbench.md (not re-measured)")


def rates_from_microbench(mb: dict) -> dict:
    """Per-instruction pipe clocks from the JSON line csrc/microbench.cu prints."""
    lop3 = mb["lop3"]
    # inside a Philox-like stream (one multiply + n LOP3): slope = LOP3 cost, intercept = what the multiply adds
    w = mb["wide_lop3"]                       # clocks for 1 multiply + (1 + NL) LOP3, NL = 0..3
    slope = (w[3] - w[1]) / 2.0
    wide_int = w[1] - 2.0 * slope             # intercept of the n >= 2 line
    return dict(ffma=mb["ffma"], ffma2=mb.get("ffma2", 2.0 * mb["ffma"]), imad=mb["imad"], imad_wide=mb["philox_block"] / 20.0, lop3=lop3, dfma=mb["dfma"],
                mufu=mb["mufu"], wide_int=wide_int, philox_block=mb["philox_block"],
                stage_a_core_row=mb["stage_a_core_row"], source="csrc/microbench.cu, run by bench.py on this box")


def U(issue, wide=0.0, imad=0.0, logic=0.0, fp64=0.0, fp32=0.0, xu=0.0):
    return dict(issue=float(issue), wide=float(wide), imad=float(imad), logic=float(logic), fp64=float(fp64),
                fp32=float(fp32), xu=float(xu))


# ---- per-unit algorithmic thread-instruction counts (profiles/r2_instruction_counts.md)
# every launched neutron: Philox block 0, words 0 and 1 only (16 wide multiplies + 2 low products survive dead-code
# elimination: counter words 1..3 are launch constants), 17.7 XOR, window compares, ballot, prefix mask, 2 POPC
STAGE_A = U(42, wide=16, imad=2, logic=22, xu=2)
# every slit-1 survivor: Philox block 1 (18.5 multiplies: two have constant inputs), 19 XOR, compaction
# (ballot, mask, 2 POPC, ring position); the classifier's 8 instructions are not counted
STAGE_B0 = U(50.5, wide=18.5, logic=30, xu=2)
# every survivor whose geometry is evaluated (Philox block 0 again is not counted)
STAGE_B = {
    "fast": U(268, logic=52, fp64=200, fp32=3, xu=13),       # slit-free box-sample instrument class (c0, c1, c2, c4)
    "general": U(307, logic=66, fp64=225, fp32=2, xu=14),    # cylinder sample, slits that may cut (c3)
}

# per detected neutron: (prologue, per node evaluation).  Rows marked (counted) are read from the executed SASS of
# the round-2 profiles (profiles/r2_instruction_counts.md); rows marked (estimate) are assembled from the counted
# pieces they share with those (Philox block: 19 multiplies + 20 XOR; sincos: 35 FP64; ...) and are not judged as
# measurements.
MODEL_COST = {
    # (counted, c0) one fp64 evaluation, all of it in the prologue
    "sphere_fp64": (U(94, wide=1, imad=1, logic=27, fp64=63, xu=2), U(0)),
    # (estimate: sphere_py_fp32 without its S(q))
    "sphere_fp32": (U(90, wide=1, imad=1, logic=22, fp64=22, fp32=30, xu=14), U(28.4, logic=1.2, fp32=27.2)),
    # (counted, c1 fp32)
    "sphere_py_fp32": (U(135.6, wide=1, imad=1, logic=24.6, fp64=22, fp32=69, xu=17), U(28.4, logic=1.2, fp32=27.2)),
    # (counted, c1 fp64)
    "sphere_py_fp64": (U(138, wide=1, imad=1, logic=32, fp64=101, fp32=1, xu=3), U(45.2, logic=15.2, fp64=30)),
    # (round-1 SASS count of the node; prologue estimate)
    # (counted, c2: executed SASS of the packed row, profiles/r2_instruction_counts.md) per tilt node 13.5 packed
    # instructions (27 FP32 operations), 0.2 scalar FP32, 0.2 logic, 1 MUFU.RCP; prologue estimate
    "cylinder_quad_fp32": (U(60, logic=10, fp64=40, xu=4), U(14.9, logic=0.2, fp32=27.2, xu=1)),
    # (counted, c3) prologue = Philox block 2 (orientation draws), three sincos of 2 pi u, frame, and the 16 outer
    # nodes (37 instructions each); inner node 34
    "cs_triaxial_iso_fp32": (U(832, wide=19, imad=18.5, logic=136, fp64=114, fp32=499, xu=47), U(19, imad=0.5, logic=2.5, fp32=28, xu=2)),   # (counted) inner node packed: 14 packed instructions = 28 FP32 operations
    # (estimate: the per-event cylinder below without its size draws)
    "cylinder_iso_fp64": (U(370, wide=37, logic=120, fp64=200, xu=6), U(0)),
    # (counted, n1) per-event sizes: Philox blocks 2 and 3 and a re-draw, two Box-Muller normals, three sin/cos of
    # pi x, sin, Lambda, the weight
    "cylinder_event_fp64": (U(562, wide=56, imad=3, logic=150, fp64=344, fp32=2, xu=7), U(0)),
    # (counted, n2) barbell, per event: everything that executes once per detected warp (size and orientation draws,
    # frame, cylinder term, weight), then 64 slice evaluations of the two end pieces (fp64 Lambda of the squared argument
    # and cosine each; recounted after the square root per slice was removed: 88 per pass of two slices)
    "barbell_event_fp64": (U(608, wide=56, imad=3, logic=155, fp64=382, fp32=3, xu=9), U(44.0, logic=5.5, fp64=38.5)),
    # (counted, n3) micelle, per event: Philox block 3, one Box-Muller normal, sphere Phi, sinc, expm1, the four terms
    "micelle_event_fp64": (U(514, wide=19, imad=2, logic=111, fp64=350, fp32=15, xu=17), U(0)),
    # (counted, n5) thin-walled hollow prism, per event: Philox blocks 2 and 3, one Box-Muller normal, the frame (three
    # sin/cos of pi x), three fp64 sine/cosine pairs of the half-side phases, the face sum
    "hollow_prism_event_fp64": (U(518, wide=38, imad=2, logic=154, fp64=313, fp32=5, xu=6), U(0)),
    # (counted, n4) charged spheres, per event: Philox block 3, one Box-Muller normal, sphere Phi, the tail term of
    # S(q) with the rotation by K/2 of the folded sum; then the 32 node PAIRS of the MSA rule, each one fp64
    # sine/cosine pair (three-step reduction, two Taylor kernels, quadrant selects) and two accumulations
    "sphere_msa_event_fp64": (U(323, wide=19, imad=2, logic=85, fp64=205, fp32=4, xu=8), U(39, logic=12, fp64=27)),
}

RESOURCES = ("issue", "imul", "int", "fp64", "xu", "fma")


def unit_sum(frac_survive, frac_geometry, frac_detect, model_key, nodes, geometry="fast"):
    """Algorithmic thread-instructions per launched neutron, by class."""
    pro, node = MODEL_COST[model_key]
    tot = {}
    for k in STAGE_A:
        tot[k] = (STAGE_A[k] + frac_survive * STAGE_B0[k] + frac_geometry * STAGE_B[geometry][k]
                  + frac_detect * (pro[k] + nodes * node[k]))
    return tot


def clocks(tot, r):
    """SMSP clocks per launched neutron-lane on each resource."""
    return dict(issue=r["ffma"] * tot["issue"],
                imul=r["imad_wide"] * tot["wide"] + r["imad"] * tot["imad"],
                int=r["lop3"] * tot["logic"] + r["wide_int"] * tot["wide"],
                fp64=r["dfma"] * tot["fp64"],
                xu=r["mufu"] * tot["xu"],
                # an FP32 operation costs half a packed instruction's time on the pair of pipes (measured: ffma2)
                fma=0.5 * (r["imad_wide"] * tot["wide"] + r["imad"] * tot["imad"]) + 0.5 * r.get("ffma2", 2.0 * r["ffma"]) * tot["fp32"])


def roofline(neutrons_per_s: float, frac_survive: float, frac_detect: float, model_key: str, nodes: int,
             sm_mhz: float = SM_MAX_MHZ, frac_geometry: float | None = None, geometry: str = "fast",
             rates: dict | None = None, sm_mhz_sampled: float | None = None, traffic=None):
    """Roofline record for bench.py.  `achieved` and `peak` are G lane-clocks/s on the binding resource
    (peak = 148 SM x 4 SMSP x 32 lanes x clock: every SMSP clock offers 32 lanes of its binding pipe)."""
    r = rates or RATES
    if frac_geometry is None:
        frac_geometry = frac_survive      # no classifier: every survivor's geometry is evaluated
    tot = unit_sum(frac_survive, frac_geometry, frac_detect, model_key, nodes, geometry)
    c = clocks(tot, r)
    pipe = max(c, key=c.get)
    peak = N_SM * SMSP_PER_SM * 32 * sm_mhz * 1e6
    achieved = neutrons_per_s * c[pipe]
    c_old = {k: v for k, v in c.items() if k != "int"}
    out = {
        "bound": "alu", "pipe": pipe,
        "achieved": achieved / 1e9, "peak": peak / 1e9, "unit": "G lane-clocks/s",
        "frac": achieved / peak,
        # the same throughput against the round-1 resource list (no logic-pipe resource)
        "frac_without_int_resource": neutrons_per_s * max(c_old.values()) / peak,
        "alg_clocks_per_neutron": {k: round(v, 2) for k, v in c.items()},
        "alg_instr_per_neutron": {k: round(v, 2) for k, v in tot.items()},
        "peak_source": (f"{N_SM} SM x {SMSP_PER_SM} SMSP x 32 lanes x {sm_mhz:.0f} MHz (maximum SM clock); clocks per "
                        f"instruction of each pipe from {r['source']}"),
        "pipe_clocks_per_warp_instruction": {k: round(float(r[k]), 3) for k in
                                             ("ffma", "ffma2", "imad", "imad_wide", "lop3", "wide_int", "dfma", "mufu") if k in r},
        "traffic": traffic,
    }
    if sm_mhz_sampled:
        out["frac_at_sampled_clock"] = out["frac"] * sm_mhz / sm_mhz_sampled
        out["sm_mhz_sampled"] = sm_mhz_sampled
    return out


def read_traffic(path: str) -> dict:
    """DRAM bytes per trace-kernel launch (dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full`
    capture per workload), read from the table of profiles/r2_dram_traffic.md: `| workload | read | written |`."""
    out = {}
    try:
        for line in open(path):
            cells = [c.strip() for c in line.strip().strip("|").split("|")]
            if len(cells) >= 3 and cells[1].replace(".", "").isdigit():
                out[cells[0]] = int(float(cells[1]) + float(cells[2]))
    except OSError:
        pass
    return out
