"""GPU parity tests proper (-m gpu): the CUDA path, called through the C ABI, against the oracle
element by element on the same seeded inputs.  Bar: bit-exact for genomes, indices, counts and
decisions; survival probabilities are produced by the same specified fp32 sequence on both sides
(so they are bit-equal, which implies north_star's 1e-6 relative bound); decisions with
|u01 - s| < 1e-6 are counted and reported in the log (`near_ties`)."""
import numpy as np
import pytest

import parity
from paper_1603_09255_b200 import workloads

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def binding():
    from paper_1603_09255_b200 import binding as b
    from paper_1603_09255_b200 import build
    build.build()          # (re)builds libspegg.so in-tree when missing or older than its sources; raises if nvcc fails
    b.load()
    return b


@pytest.mark.parametrize("which,scale,grid,steps", [
    (1, 1.0, None, 6),        # C1 at full size
    (2, 0.05, None, 3),       # C2: 5,000 individuals, 4 chromosomes
    (3, 0.02, None, 3),       # C3: 20,000 individuals: several tiles and a ragged tail
    (4, 0.004, None, 3),      # C4: two species
    (5, 0.03, (6, 5), 3),     # C5: 30 patches on a 6x5 torus
])
def test_per_step_parity_debug(oracle_mod, binding, which, scale, grid, steps):
    cfg = workloads.config(which, scale=scale, grid=grid)
    parity.per_step_parity(oracle_mod, binding, cfg, steps, debug=True)


@pytest.mark.parametrize("which,scale,grid,steps", [
    (1, 1.0, None, 4), (3, 0.013, None, 3), (5, 0.03, (4, 4), 2), (4, 0.004, None, 2), (2, 0.03, None, 2)])
def test_per_step_parity_fast_path(oracle_mod, binding, which, scale, grid, steps):
    # debug off: the production (fused where available) kernels; state and log must still match
    cfg = workloads.config(which, scale=scale, grid=grid)
    parity.per_step_parity(oracle_mod, binding, cfg, steps, debug=False)


SEEDS = [1, 2, 3, 0x9E3779B97F4A7C15]     # seeds 1-3; the last one has a non-zero HIGH key word


@pytest.mark.parametrize("seed", SEEDS)
@pytest.mark.parametrize("which,scale,grid,debug", [
    (3, 0.013, None, False),      # the fused C3 kernels (the ones bench.py times)
    (3, 0.006, None, True),
    (2, 0.02, None, False), (5, 0.02, (4, 3), False), (4, 0.003, None, False), (1, 1.0, None, True),
])
def test_per_step_parity_seeds(oracle_mod, binding, which, scale, grid, debug, seed):
    """Every configuration on other seeds than its own, including a 64-bit seed whose high word is
    not zero: Philox key word k1 = seed >> 32 (R3) reaches the kernels through the host-built round
    keys, and a dropped or swapped high word would pass every test that only uses small seeds."""
    cfg = workloads.config(which, scale=scale, grid=grid, seed=seed)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=debug)


def _c3(scale, **kw):
    cfg = workloads.config(3, scale=scale)
    cfg["species"][0].update(kw)
    return cfg


def _assert_fused(sim):
    assert sim.launches_per_step() == 2, "configuration left the fused two-kernel step"


def _free_run(oracle_mod, binding, cfg, steps, chunks=1, fused=True):
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    if fused is not None:
        assert (sim.launches_per_step() == 2) == fused
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(chunks):
        orc.step(steps)
        sim.step(steps)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
        assert sim.status() == orc.flags
    sim.close()
    return orc


@pytest.mark.parametrize("capacity", [24576, 24001])
def test_fused_path_capacity_overflow(oracle_mod, binding, capacity):
    """OVERFLOW on the fused C3 kernels (k_scan_fused truncates M_t at the capacity, k_fused_bit_f stops
    at it): K = 1e9 keeps lambda at 2, so M_t > capacity in every step; the second capacity is not a
    multiple of the 32-row slab.  Per step from the oracle's state, then free-running."""
    cfg = _c3(0.02, K=1e9, capacity=capacity)
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=False)
    orc = _free_run(oracle_mod, binding, cfg, 3)
    assert all(e["flags"] & 1 and e["m_t"] == capacity for e in orc.log(0))


def test_fused_path_unstaged_mother_ranges(oracle_mod, binding):
    """k_scan_fused stages the mother[] words of a 1,024-row range in shared memory when the range has at
    most 4,096 offspring and stores them directly otherwise: lambda = 8 gives ~8,000 per range (asserted
    from the oracle's fecundities), and the second step overflows the capacity on the same path."""
    cfg = _c3(0.02, fec_a=8.0, K=1e9)
    cfg["species"][0]["capacity"] = 10 * cfg["n0"][0] // 1024 * 1024
    orc = oracle_mod.Oracle(cfg)
    parity.load_initial(orc, cfg)
    orc.step(1)
    f = orc.debug(0)["f"].astype(np.int64)
    per_range = np.add.reduceat(f, np.arange(0, len(f), 1024))
    assert per_range.max() > 4096
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)
    orc = _free_run(oracle_mod, binding, cfg, 2)
    assert orc.log(0)[0]["flags"] == 0 and orc.log(0)[1]["flags"] & 1


@pytest.mark.parametrize("kw", [
    dict(xover_mean=[0.0, 0.0, 0.0, 0.0]),                 # no crossover tables at all: whole parental haplotypes
    dict(xover_mean=[0.3, 1.0, 3.0, 4.0]),                 # most chromosomes draw > 2 crossovers: the fix-up queue overflows in every chunk
    dict(xover_mean=[12.0, 0.0, 20.0, 1.0]),               # crossover draws from several RECOMB blocks of a chromosome
    dict(mu=1e-3),                                         # L mu = 1.02: several mutations per gamete (MUT blocks k > 0), both gametes
    dict(mu=0.0),                                          # L mu = 0: an empty mutation table (no gamete ever mutates)
    dict(gaussian=dict(theta0=0.5, dtheta=0.01, omega=1.5, theta_patch=None)),   # moving optimum
    dict(gaussian=None),                                   # no selection: everybody survives, all slabs full
    dict(gaussian=dict(theta0=30.0, dtheta=0.0, omega=0.5, theta_patch=None)),   # nobody survives: extinction on the fused path
])
def test_fused_path_genetics_and_selection(oracle_mod, binding, kw):
    """Non-default genetics and selection on the fused C3 kernels (bench.py's kernels): per step from
    the oracle's state, then a free-running trajectory."""
    cfg = _c3(0.012, **kw)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)
    _free_run(oracle_mod, binding, cfg, 4, chunks=2)


@pytest.mark.parametrize("n0", [1, 31, 33, 1023, 1025, 2049, 4097])
def test_fused_path_ragged_sizes(oracle_mod, binding, n0):
    """Ragged tails of the fused kernels: one adult, a 32-row slab minus / plus one, a 1,024-row scan
    range minus / plus one, two and four ranges plus one; and an empty population stays empty."""
    cfg = _c3(0.01, fec_a=3.0, K=float(max(n0, 8)), capacity=max(4 * n0, 256))
    cfg["n0"] = [n0]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=False)
    _free_run(oracle_mod, binding, cfg, 6)
    sim = binding.Sim(cfg, debug=False)
    _assert_fused(sim)
    sim.write_state(0, workloads.initial_rows(cfg, 0)[:0], None, 0)
    sim.step(2)
    assert sim.n(0) == 0 and (sim.status() & 2)
    sim.close()


def test_unequal_chromosomes_leave_the_fused_kernel(oracle_mod, binding):
    """k_fused_bit_f<4, 8> is written for four chromosomes of 256 loci; any other split of 1,024 loci must
    run the general pipeline (and still match the oracle on the production path)."""
    cfg = _c3(0.01, chrom_len=[512, 256, 128, 128], xover_mean=[2.0, 1.0, 0.5, 0.5])
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)
    _free_run(oracle_mod, binding, cfg, 5, fused=False)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=True)


def test_read_state_keeps_the_debug_view(oracle_mod, binding):
    """spegg_read_state stages in the idle population buffer, so the debug view of the last step is
    still intact after it; spegg_read_log spans the ring wrap in two copies and `last=n` reads n entries."""
    cfg = workloads.config(2, scale=0.02)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=True, log_capacity=8)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    orc.step(11)
    sim.step(11)
    parity.assert_state_equal(sim, orc, cfg)                       # read_state first ...
    parity.assert_debug_equal(sim.read_debug(0), orc.debug(0), cfg["species"][0])   # ... the view is unchanged
    assert sim.read_log(0, last=8) == orc.log(0)[-8:]             # entries 3..10 of a ring of 8: wraps
    assert sim.read_log(0, last=1) == orc.log(0)[-1:]
    with pytest.raises(binding.SpeggError) as e:
        sim.read_log(0)                                            # entries 0..2 were overwritten
    assert e.value.code == binding.ERANGE
    sim.close()


@pytest.mark.parametrize("which,scale,grid,steps", [(1, 1.0, None, 100), (3, 0.01, None, 40), (5, 0.02, (5, 4), 25),
                                                    (4, 0.003, None, 25), (2, 0.02, None, 30)])
def test_free_running_trajectory(oracle_mod, binding, which, scale, grid, steps):
    # no re-seeding: because every decision is taken in identical arithmetic the whole trajectory
    # (N_t, M_t, sums of phenotypes, genomes) must stay bit-identical
    cfg = workloads.config(which, scale=scale, grid=grid)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    orc.step(steps)
    sim.step(steps)
    for s in range(len(cfg["species"])):
        parity.assert_logs_equal(sim.read_log(s), orc.log(s), tag="species %d" % s)
    parity.assert_state_equal(sim, orc, cfg)
    assert sim.step_counter == orc.step_counter == steps
    sim.close()


def test_step_n_equals_n_steps_and_checkpoint(binding):
    cfg = workloads.config(3, scale=0.01)
    a = binding.Sim(cfg)
    b = binding.Sim(cfg)
    parity.load_initial(a, cfg)
    parity.load_initial(b, cfg)
    a.step(4)
    b.step(1); b.step(1)
    rows, ps, _ = b.read_state(0)
    c = binding.Sim(cfg)                     # resume from a checkpoint in a fresh handle
    c.write_state(0, rows, None, 2)
    c.step(2)
    ra, _, za = a.read_state(0)
    rc, _, zc = c.read_state(0)
    assert np.array_equal(ra, rc) and np.array_equal(za, zc)
    # write_state(read_state()) is the identity
    c.write_state(0, rc, None, 4)
    assert np.array_equal(c.read_state(0)[0], rc)
    for s in (a, b, c):
        s.close()


def test_overflow_and_extinction(oracle_mod, binding):
    cfg = workloads.config(1)
    cfg["species"][0]["capacity"] = 1024
    cfg["species"][0]["K"] = 1e9
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=True)
    sim = binding.Sim(cfg)
    parity.load_initial(sim, cfg)
    sim.step(1)
    assert sim.status() & 1
    sim.close()
    cfg = workloads.config(1)
    cfg["species"][0]["fec_a"] = 0.0
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    orc.step(3); sim.step(3)
    parity.assert_logs_equal(sim.read_log(0), orc.log(0))
    assert sim.n(0) == 0 and sim.status() == orc.flags and sim.status() & 2
    sim.close()


def test_empty_population_and_device_rows(binding):
    import torch
    cfg = workloads.config(3, scale=0.004)
    sim = binding.Sim(cfg)
    sim.step(2)                               # nothing loaded: N = 0, steps are no-ops
    assert sim.n(0) == 0
    rows = workloads.initial_rows(cfg, 0)
    dev = torch.from_numpy(rows.view(np.int32)).cuda()
    sim.write_state(0, dev, None, 0)          # rows given as a DEVICE pointer
    other = binding.Sim(cfg)
    other.write_state(0, rows, None, 0)
    sim.step(2); other.step(2)
    assert np.array_equal(sim.read_state(0)[0], other.read_state(0)[0])
    sim.close(); other.close()


def test_bad_parameters_are_rejected(binding):
    cfg = workloads.config(3, scale=0.001)
    cfg["species"][0]["chrom_len"] = [100, 924]   # bit chromosomes must be word-aligned
    cfg["species"][0]["xover_mean"] = [1.0, 1.0]
    with pytest.raises(binding.SpeggError):
        binding.workspace_bytes(cfg)
    cfg = workloads.config(1)
    cfg["species"][0]["mu"] = 1.5
    with pytest.raises(binding.SpeggError):
        binding.workspace_bytes(cfg)


# ---- BASELINE.json's FULL sizes, in the launch configuration bench.py times (debug off, the
# production kernels, the captured graph).  The oracle finishes a full-size step in seconds
# (C3 ~6 s, C4 ~9 s, C5 ~17 s per step), so the comparison is complete -- every row of the next
# generation, every log field -- rather than sampled.
@pytest.mark.parametrize("which,steps", [(3, 3), (2, 6), (4, 3), (5, 3)])
def test_full_size_bench_configuration(oracle_mod, binding, which, steps):
    cfg = workloads.config(which)                     # scale 1.0: N0, K, capacity as benchmarked
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    for s in range(len(cfg["species"])):
        rows = workloads.initial_rows(cfg, s)
        ps = workloads.initial_patch_start(cfg, s)
        orc.write_state(s, rows, ps, 0)
        sim.write_state(s, rows, ps, 0)
        del rows
    orc.step(steps)
    sim.step(steps)                                   # free-running: step t+1 consumes the GPU's own step t
    for s in range(len(cfg["species"])):
        parity.assert_logs_equal(sim.read_log(s), orc.log(s), tag="C%d species %d" % (which, s))
    parity.assert_state_equal(sim, orc, cfg, tag="C%d full size" % which)
    assert sim.status() == orc.flags
    sim.close()


def _q10_variant(n_loci, chrom_len, r_within, mu, n0=3000):
    """C1 with another genetic architecture: exercises the lane layouts of the vectorised q10
    gamete kernel (L / 8 lanes per gamete) and, with a high mutation rate, the phenotype
    correction applied by the mutation kernel."""
    cfg = workloads.config(1, scale=n0 / 1000.0)
    sp = cfg["species"][0]
    sp.update(n_loci=n_loci, chrom_len=list(chrom_len), r=workloads._interval_r(list(chrom_len), r_within), mu=mu)
    return cfg


@pytest.mark.parametrize("n_loci,chrom_len,r,mu", [
    (8, [8], 0.5, 0.02),              # one lane per gamete pair of blocks: 16 offspring per warp
    (32, [16, 16], 0.1, 0.05),        # 4 lanes per gamete, many mutations per step
    (256, [256], 0.02, 1e-3),         # 32 lanes per gamete: the two gametes in successive passes
    (128, [100, 28], 0.3, 1e-2),      # chromosome boundary inside a lane's 8 loci
    (24, [24], 0.25, 1e-2),           # not a power of two: the plain kernels
])
def test_q10_lane_layouts_free_running(oracle_mod, binding, n_loci, chrom_len, r, mu):
    cfg = _q10_variant(n_loci, chrom_len, r, mu)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(3):            # compare along the way too, so that a first divergence is localised
        orc.step(5)
        sim.step(5)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    sim.close()


def test_sweep_of_unlinked_patches(oracle_mod, binding):
    """S6: with m = 0 the patches are independent replicates
    with their own parameters.  Parity with the oracle, and the metamorphic properties SURVEY.md
    section 4 lists: no individual ever changes patch, and an emptied patch stays empty."""
    cfg = workloads.config(6, scale=0.01, grid=(6, 1))
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=True)
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=False)
    rows = workloads.initial_rows(cfg, 0)
    ps = workloads.initial_patch_start(cfg, 0).astype(np.int64)
    a, b = ps[2], ps[3]                                  # patch 2 starts empty
    rows = np.concatenate([rows[:a], rows[b:]])
    ps2 = ps.copy()
    ps2[3:] -= b - a
    ps2 = ps2.astype(np.uint32)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=True)
    for o in (orc, sim):
        o.write_state(0, rows, ps2, 0)
    for t in range(4):
        before = sim.read_state(0)[1].astype(np.int64)   # patch_start of the adults
        orc.step(1)
        sim.step(1)
        d = sim.read_debug(0)
        natal = np.searchsorted(before, d["mother"].astype(np.int64), side="right") - 1
        assert np.array_equal(natal, d["dest"].astype(np.int64)), "an offspring left its natal patch"
        parity.assert_debug_equal(d, orc.debug(0), cfg["species"][0], tag="step %d" % t)
    parity.assert_state_equal(sim, orc, cfg)
    after = sim.read_state(0)[1].astype(np.int64)
    sizes = np.diff(after)
    assert sizes[2] == 0 and (np.delete(sizes, 2) > 0).all()
    sim.close()


@pytest.mark.parametrize("which,scale,rho", [(2, 0.05, 0.3), (1, 2.0, 1.0), (3, 0.01, 0.75), (5, 0.02, 0.25)])
def test_residual_phenotype_noise(oracle_mod, binding, which, scale, rho):
    """R17, eq. S2-14: residual phenotype noise.  Per-step parity of every
    intermediate (debug), then a free-running trajectory on the production kernels (for the bit
    configuration the NOISE instantiation of the fused kernel: test_fused_path_residual_noise)."""
    cfg = workloads.config(which, scale=scale, grid=(4, 3) if which == 5 else None)
    cfg["species"][0]["resid_sd"] = rho
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    orc.step(8)
    sim.step(8)
    parity.assert_logs_equal(sim.read_log(0), orc.log(0))
    parity.assert_state_equal(sim, orc, cfg)
    sim.close()


@pytest.mark.parametrize("which,scale,sA,rho", [(1, 1.0, 0.975, 0.0), (2, 0.04, 0.6, 0.0), (3, 0.008, 0.5, 0.0),
                                                 (2, 0.03, 0.8, 0.2)])
def test_overlapping_generations(oracle_mod, binding, which, scale, sA, rho):
    """R18: adults stay alive with probability s_A w(z); the next generation is
    the staying adults followed by the surviving offspring.  Per-step parity of every intermediate
    (debug), then a free-running trajectory on the production kernels."""
    cfg = workloads.config(which, scale=scale)
    sp = cfg["species"][0]
    sp["adult_survival"] = sA
    sp["resid_sd"] = rho
    sp["capacity"] = 4 * sp["capacity"]          # generations pile up: N* = K (2 w / (1 - s_A w) - 1)
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(6)
        sim.step(6)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()


def test_overlapping_generations_room_for_offspring(oracle_mod, binding):
    # M_t <= capacity - N_t: the overflow flag and the truncation agree with the oracle
    cfg = workloads.config(1, scale=1.5)
    sp = cfg["species"][0]
    sp.update(adult_survival=0.9, K=1e9, capacity=2048)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=True)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)


@pytest.mark.parametrize("which,scale,v,grid,extra", [
    (1, 1.0, 2.0, None, {}),                        # C1, strong preference
    (2, 0.06, 1.0, None, {}),                       # C2: 6,000 adults = several weight tiles and a ragged tail
    (2, 0.04, -3.0, None, {"resid_sd": 0.2}),       # preference for small mates, with residual noise (same SCALAR block)
    (3, 0.012, 0.5, None, {}),                      # bit genome: the general pipeline in debug, the MATE instantiation of the fused kernel in production
    (5, 0.03, 1.5, (5, 4), {}),                     # patches: the father comes from the mother's patch
    (2, 0.04, 1.0, None, {"adult_survival": 0.6}),  # with overlapping generations
    (1, 1.0, 400.0, None, {}),                      # clamp in play, most integer weights are 0
])
def test_shared_preference_mating(oracle_mod, binding, which, scale, v, grid, extra):
    """R19 (eq. S2-10): the father is drawn with probability
    proportional to exp(v_m z) by integer running sum + search.  Per-step parity of every
    intermediate including the running sum (debug), then a free-running trajectory on the
    production kernels."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["mate_skew"] = v
    sp.update(extra)
    if "adult_survival" in extra:
        sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(5)
        sim.step(5)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()


def test_shared_preference_mating_full_size(oracle_mod, binding):
    """R19 at C2's full size (100,000 adults, ~100 weight tiles) on the production kernels: one step
    from the oracle's state, fathers compared through the offspring that survive (state + log)."""
    cfg = workloads.config(2)
    cfg["species"][0]["mate_skew"] = 1.0
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)


@pytest.mark.parametrize("scale,E,v,extra", [
    (0.004, 3, 0.15, {}),                     # C4 shape: 4,000 prey, 400 consumers, three meetings each
    (0.004, 1, 0.4, {}),                      # one meeting, strong
    (0.004, 1, 1.0, {}),                      # so strong that the consumers overshoot and go extinct at step 2
    (0.003, 16, 0.05, {}),                    # the maximum: eight SCALAR blocks per newborn
    (0.004, 4, 0.3, {"resid_sd": 0.5}),       # with residual phenotype noise on the newborn's trait
    (0.004, 2, 2.0, {"mate_skew": 1.0}),      # with weighted fathers (both use later SCALAR blocks)
])
def test_individual_encounters(oracle_mod, binding, scale, E, v, extra):
    """R20 (eq. S3-2): each newborn meets E uniformly drawn consumers;
    captures are credited to the consumer met.  Per-step parity of every intermediate of both
    species (debug), then a free-running trajectory on the production kernels."""
    cfg = workloads.config(4, scale=scale)
    cfg["species"][0]["predation"].update(encounters=E, attack=v)
    cfg["species"][0].update(extra)
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(6)
        sim.step(6)
        for s in range(2):
            parity.assert_logs_equal(sim.read_log(s), orc.log(s), tag="species %d" % s)
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    assert sum(e["captures"] for e in orc.log(0)) > 0
    sim.close()


@pytest.mark.parametrize("which,scale,grid,extra", [
    (1, 1.0, None, {}),                                   # C1, uniform over the males
    (2, 0.06, None, {"mate_skew": 1.5}),                  # C2, R19's weights among the males
    (3, 0.012, None, {}),                                 # bit genome on the general pipeline
    (5, 0.03, (5, 4), {"mate_skew": -1.0}),               # patches: males of the mother's patch
    (2, 0.04, None, {"adult_survival": 0.6}),             # overlapping generations: staying adults keep their sex
    (1, 1.0, None, {"resid_sd": 0.5, "mate_skew": 3.0}),
])
def test_separate_sexes(oracle_mod, binding, which, scale, grid, extra):
    """R21 (eqs. S2-9/S2-10): only females lay eggs, only males father them, the sex
    travels with the individual.  Per-step parity of every intermediate incl. the offspring's sexes
    and the running sum (debug), then a free-running trajectory on the production kernels (state,
    sexes and log)."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["separate_sexes"] = 1
    sp["fec_a"] = 2.0 * sp["fec_a"]            # half the adults lay eggs
    sp.update(extra)
    if "adult_survival" in extra:
        sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(5)
        sim.step(5)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags and orc.n(0) > 0
    sex = sim.read_sex(0)
    assert 0 < sex.sum() < len(sex)
    sim.close()


def test_sex_io_errors_and_roundtrip(binding):
    """spegg_write_sex / spegg_read_sex: ESTATE without separate sexes, ERANGE for a wrong count,
    everybody female after spegg_write_state, exact round trip, encounters need sel_predation."""
    cfg = workloads.config(1)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(sim, cfg)
    with pytest.raises(binding.SpeggError) as e:
        sim.write_sex(0, np.zeros(cfg["n0"][0], np.uint8))
    assert e.value.code == binding.ESTATE
    sim.close()
    cfg["species"][0]["separate_sexes"] = 1
    sim = binding.Sim(cfg, debug=False)
    sim.write_state(0, workloads.initial_rows(cfg, 0), None, 0)
    assert (sim.read_sex(0) == 0).all()
    with pytest.raises(binding.SpeggError) as e:
        sim.write_sex(0, np.zeros(cfg["n0"][0] - 1, np.uint8))
    assert e.value.code == binding.ERANGE
    sex = workloads.initial_sex(cfg, 0)
    sim.write_sex(0, sex * 7)                    # any non-zero byte is male
    assert np.array_equal(sim.read_sex(0), sex)
    sim.close()
    cfg = workloads.config(4, scale=0.002)
    cfg["species"][1]["encounters"] = 3          # not a predation parameter of the consumer itself
    cfg["species"][0]["predation"]["encounters"] = 17
    with pytest.raises(binding.SpeggError):
        binding.workspace_bytes(cfg)


@pytest.mark.parametrize("which,variant", [(4, "encounters"), (5, "sexes+mating")])
def test_full_size_widenings(oracle_mod, binding, which, variant):
    """The widenings at BASELINE.json's full sizes on the production kernels (the launch configuration
    `bench.py --variant` times): one step, every row, sex and log field compared with the oracle."""
    cfg = workloads.config(which)
    sp = cfg["species"][0]
    if variant == "encounters":
        sp["predation"].update(encounters=3, attack=0.1)      # R20: 1.3 M newborns x 3 meetings with 100,000 consumers
    else:
        sp.update(separate_sexes=1, mate_skew=1.0)            # R21 + R19 in 4,096 patches: ~4,600 weight tiles
        sp["fec_a"] = 2.0 * sp["fec_a"]
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    orc.step(1)
    sim.step(1)
    for s in range(len(cfg["species"])):
        parity.assert_logs_equal(sim.read_log(s), orc.log(s), tag="C%d+%s species %d" % (which, variant, s))
    parity.assert_state_equal(sim, orc, cfg, tag="C%d+%s full size" % (which, variant))
    assert sim.status() == orc.flags
    sim.close()


@pytest.mark.parametrize("which,scale", [(3, 1.0), (2, 1.0), (5, 0.1), (4, 0.05)])
def test_sixteen_step_graph_equals_single_steps(binding, which, scale):
    """spegg_step(n) replays a sixteen-step graph for long runs (the launch configuration bench.py
    times: consecutive steps' kernels overlap through programmatic edges) and a one-step graph for
    the remainder.  Both must produce the same trajectory: 35 steps in one call against 35 calls of
    one step, at C3's full size -- whose first steps are checked against the oracle in
    test_full_size_bench_configuration -- state and log compared bit for bit."""
    cfg = workloads.config(which, scale=scale)
    a = binding.Sim(cfg, debug=False)
    b = binding.Sim(cfg, debug=False)
    parity.load_initial(a, cfg)
    parity.load_initial(b, cfg)
    a.step(35)
    for _ in range(35):
        b.step(1)
    for s in range(len(cfg["species"])):
        assert a.read_log(s) == b.read_log(s)
        ra, pa, za = a.read_state(s)
        rb, pb, zb = b.read_state(s)
        assert np.array_equal(ra, rb) and np.array_equal(pa, pb) and np.array_equal(za, zb)
    assert a.status() == b.status() and a.step_counter == b.step_counter == 35
    a.close()
    b.close()


@pytest.mark.parametrize("n0", [1, 31, 33, 1023, 1025, 2049])
def test_mating_paths_ragged_sizes(oracle_mod, binding, n0):
    """Ragged tails of the mating path: one adult, a block of 32 minus / plus one, a weight tile of
    1,024 minus / plus one, two tiles plus one -- separate sexes with weighted fathers, per-step
    parity of every intermediate; and an empty population stays empty."""
    cfg = workloads.config(1, scale=n0 / 1000.0)
    cfg["n0"] = [n0]
    sp = cfg["species"][0]
    sp.update(separate_sexes=1, mate_skew=2.0, K=float(max(n0, 8)), capacity=max(4 * n0, 256))
    sp["fec_a"] = 4.0
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=False)
    sim = binding.Sim(cfg, debug=False)
    sim.write_state(0, workloads.initial_rows(cfg, 0)[:0], None, 0)
    sim.step(2)
    assert sim.n(0) == 0 and (sim.status() & 2) and len(sim.read_sex(0)) == 0
    sim.close()


@pytest.mark.parametrize("which,scale,rho,grid,extra", [
    (1, 1.0, 0.5, None, {}),
    (2, 0.05, 2.0, None, {"fec_a": 6.0}),                     # up to a dozen eggs drawn per adult: several FEC blocks
    (3, 0.01, 0.02, None, {}),                                # bit genome on the general pipeline
    (5, 0.03, 1.0, (5, 4), {}),                               # patches
    (2, 0.04, 1.0, None, {"separate_sexes": 1, "mate_skew": 1.0, "adult_survival": 0.5, "fec_a": 6.0}),
])
def test_fecundity_cost(oracle_mod, binding, which, scale, rho, grid, extra):
    """R22 (eq. S3-3): each egg of adult i is laid with probability exp(-rho z_i^2).
    Per-step parity of every intermediate (debug), then a free-running trajectory on the production
    kernels."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["fec_cost"] = rho
    sp.update(extra)
    if "adult_survival" in extra:
        sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(5)
        sim.step(5)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()


def test_resource_with_cost_meets_consumers(oracle_mod, binding):
    """The S3 community in one piece: the resource pays the fecundity cost of its defence trait (R22),
    its newborns meet consumers individually (R20), the consumers' fecundity follows their captures."""
    cfg = workloads.config(4, scale=0.004)
    cfg["species"][0]["predation"].update(encounters=3, attack=0.1)
    cfg["species"][0]["fec_cost"] = 0.05
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    parity.per_step_parity(oracle_mod, binding, cfg, 4, debug=False)


@pytest.mark.parametrize("which,scale,a,grid,extra", [
    (1, 1.0, 2.0, None, {}),
    (2, 0.05, 1.0, None, {}),
    (2, 0.04, 30.0, None, {"resid_sd": 0.3}),              # choosy: most eggs use all 8 candidates
    (3, 0.01, 0.5, None, {}),                              # bit genome on the general pipeline
    (5, 0.03, 1.5, (5, 4), {}),                            # candidates from the mother's patch
    (2, 0.04, 1.0, None, {"adult_survival": 0.5, "fec_cost": 0.2}),
])
def test_assortative_mating(oracle_mod, binding, which, scale, a, grid, extra):
    """R23: candidate fathers accepted with probability exp(-a (z_c - z_m)^2).  Per-step
    parity of every intermediate (debug), then a free-running trajectory on the production kernels."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["assort"] = a
    sp.update(extra)
    if "adult_survival" in extra:
        sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(5)
        sim.step(5)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()
    bad = workloads.config(1)
    bad["species"][0].update(assort=1.0, mate_skew=1.0)     # the two mating rules exclude each other
    with pytest.raises(binding.SpeggError):
        binding.workspace_bytes(bad)


@pytest.mark.parametrize("which,scale,v,grid,extra", [
    (1, 1.0, 2.0, None, {}),                                              # C1, strong skew
    (2, 0.06, 1.0, None, {}),                                             # C2: several weight tiles and a ragged tail
    (2, 0.04, -2.0, None, {"mate_skew": 1.5}),                            # both parents weighted, opposite signs
    (3, 0.012, 0.5, None, {}),                                            # bit genome: leaves the fused kernel
    (5, 0.03, 1.5, (5, 4), {}),                                           # patches: the mother comes from the laying patch
    (5, 0.03, 1.0, (5, 4), {"separate_sexes": 1, "mate_skew": 1.0}),      # only females mother, only males father
    (2, 0.04, 1.0, None, {"adult_survival": 0.6, "assort": 2.0}),         # overlapping generations; R23 reads the NEW mother's value
    (1, 1.0, 400.0, None, {}),                                            # clamp in play, most integer weights are 0
])
def test_weighted_mothers(oracle_mod, binding, which, scale, v, grid, extra):
    """R24 (eq. S2-9): the mother of each egg is drawn with probability proportional
    to exp(v_f z) among the adults of the patch that laid it.  Per-step parity of every intermediate
    including the running sum and the reassigned mother[] (debug), then a free-running trajectory
    on the production kernels."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["mother_skew"] = v
    sp.update(extra)
    if "adult_survival" in extra:
        sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(5)
        sim.step(5)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()


def test_weighted_mothers_full_size_and_rejections(oracle_mod, binding):
    """R24 at C2's full size on the production kernels (two steps from the oracle's state), and the
    combinations the reading excludes."""
    cfg = workloads.config(2)
    cfg["species"][0]["mother_skew"] = 1.0
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)
    bad = workloads.config(1)
    bad["species"][0].update(mother_skew=1.0, fec_cost=0.5)
    with pytest.raises(Exception):
        binding.Sim(bad, debug=False)


@pytest.mark.parametrize("which,scale,grid,sA,extra", [
    (5, 0.03, (5, 4), 0.6, {}),                                   # C5 shape: dispersal between patches, adults stay put
    (5, 0.02, (4, 4), 0.9, {"resid_sd": 0.2}),                    # long-lived adults, residual noise on the juveniles
    (6, 0.004, (6, 1), 0.5, {}),                                  # S6 + overlap: case study 1's shape
    (5, 0.03, (3, 3), 0.7, {"separate_sexes": 1, "mate_skew": 1.0, "mother_skew": 1.0}),   # sexes travel with the staying adults
    (5, 0.03, (2, 1), 0.6, {}),                                   # two patches: both neighbours coincide
    (6, 0.1, (4, 1), 0.5, {}),                                    # few large patches: 17 segments per patch in the compaction
    (5, 3.0, (3, 2), 0.0, {}),                                    # the segments without overlapping generations (3,000 per patch, dispersal)
])
def test_overlapping_generations_in_patches(oracle_mod, binding, which, scale, grid, sA, extra):
    """R18 in patch mode: in every patch the staying adults (their own patch's
    optimum, rows unchanged) come before the surviving offspring that land there.  Per-step parity of
    every intermediate (debug: rows moved) and on the production kernels (index only: the staying
    adults' rows copied behind the offspring rows), then a free-running trajectory."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["adult_survival"] = sA
    sp.update(extra)
    sp["capacity"] = 6 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for _ in range(2):
        orc.step(6)
        sim.step(6)
        for s_ in range(len(cfg["species"])):
            parity.assert_logs_equal(sim.read_log(s_), orc.log(s_))
        parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()


def test_overlapping_generations_in_patches_full_size(oracle_mod, binding):
    """S6 at the paper's size (16 patches x 50,000) with overlapping generations, production
    kernels: two steps from the oracle's state."""
    cfg = workloads.config(6)
    sp = cfg["species"][0]
    sp["adult_survival"] = 0.5
    sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)


@pytest.mark.parametrize("scale,v,extra", [
    (0.012, 0.5, {}),                           # 12,000 adults: several scan ranges, weight tiles and a ragged tail
    (0.004, -2.0, {"dtheta": 0.01}),            # preference for small mates, moving optimum
    (0.002, 400.0, {}),                         # clamp in play: most weights are 0
])
def test_fused_path_weighted_father(oracle_mod, binding, scale, v, extra):
    """R19 on the fused C3 kernels (the MATE instantiation of k_fused_bit_f: father by running sum +
    search in the scalar stage, the genetic value left in zrow[] for the next step's weights).
    Production kernels only (debug runs the general pipeline): per-step from the oracle's state, then
    a free-running trajectory -- the second step onward reads the zrow[] the kernel itself wrote."""
    cfg = _c3(scale, mate_skew=v, **{k: x for k, x in extra.items() if k != "dtheta"})
    if "dtheta" in extra:
        cfg["species"][0]["gaussian"]["dtheta"] = extra["dtheta"]
    sim = binding.Sim(cfg, debug=False)
    assert sim.launches_per_step() == 4, "scan + weights + running sum + gamete kernel"
    sim.close()
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=False)
    _free_run(oracle_mod, binding, cfg, 6, chunks=2, fused=None)


@pytest.mark.parametrize("scale,rho,extra", [
    (0.013, 0.75, {}),                          # several ranges and a ragged tail
    (0.004, 4.0, {"dtheta": 0.02}),             # wide noise (256 quanta of sd), moving optimum
    (0.006, 0.25, {"mate_skew": 2.0}),          # with the weighted father: both extra draws come from SCALAR block 1
    (0.002, 0.02, {}),                          # sd of about one quantum: the table is three entries wide
])
def test_fused_path_residual_noise(oracle_mod, binding, scale, rho, extra):
    """R17 on the fused C3 kernels (the NOISE instantiations of k_fused_bit_f: one more SCALAR block and a
    table search in the survival stage; sums, zrow[] and the stored rows keep the genetic value).
    Production kernels only (debug runs the general pipeline): the configuration must STAY on the fused
    two-kernel step; per-step parity from the oracle's state, then a free-running trajectory, then the
    same trajectory in one 35-step call (16 + 16 + 2 + 1 graphs)."""
    cfg = _c3(scale, resid_sd=rho, **{k: x for k, x in extra.items() if k != "dtheta"})
    if "dtheta" in extra:
        cfg["species"][0]["gaussian"]["dtheta"] = extra["dtheta"]
    sim = binding.Sim(cfg, debug=False)
    assert sim.launches_per_step() == (4 if "mate_skew" in extra else 2), "residual noise left the fused step"
    sim.close()
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=False)
    _free_run(oracle_mod, binding, cfg, 6, chunks=2, fused=None)
    _free_run(oracle_mod, binding, cfg, 35, chunks=1, fused=None)


@pytest.mark.parametrize("which,scale,grid,extra", [
    (1, 1.0, None, {}),                                                    # C1: uniform mate, one per mother
    (2, 0.05, None, {"mate_skew": 1.5}),                                   # the pair drawn by R19's weights
    (5, 0.03, (5, 4), {"separate_sexes": 1}),                              # patches + sexes: one male per female per step
    (2, 0.04, None, {"assort": 2.0, "adult_survival": 0.6}),               # assortative pairs, staying mothers re-pair every step
    (3, 0.012, None, {"mother_skew": 1.0}),                                # bit genome (general pipeline); the pair belongs to the DRAWN mother
])
def test_monogamy(oracle_mod, binding, which, scale, grid, extra):
    """R25 ("monogamy or polygynandry"): the father's draws are addressed by the mother, so a
    clutch has one father.  Per-step parity of every intermediate (debug), per-step parity on the
    production kernels, then a free-running trajectory."""
    cfg = workloads.config(which, scale=scale, grid=grid)
    sp = cfg["species"][0]
    sp["monogamy"] = 1
    sp.update(extra)
    if "adult_survival" in extra:
        sp["capacity"] = 4 * sp["capacity"]
    parity.per_step_parity(oracle_mod, binding, cfg, 3, debug=True)
    parity.per_step_parity(oracle_mod, binding, cfg, 2, debug=False)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    orc.step(8)
    sim.step(8)
    parity.assert_logs_equal(sim.read_log(0), orc.log(0))
    parity.assert_state_equal(sim, orc, cfg)
    assert sim.status() == orc.flags
    sim.close()


def _random_cfg(rng):
    """A random small configuration: genome, structure and a random subset of the widenings that the
    validation accepts together (seeded; the combinations no hand-written case lists)."""
    grid = [None, None, (2, 1), (3, 2), (4, 4)][rng.integers(0, 5)]
    kind = "q10" if (grid is not None or rng.random() < 0.7) else "bit"
    if kind == "bit":
        cfg = workloads.config(3, scale=float(rng.choice([0.002, 0.004, 0.0065])))
        sp = cfg["species"][0]
        if rng.random() < 0.5:
            sp["xover_mean"] = [float(x) for x in rng.choice([0.0, 0.3, 1.0, 2.5], size=4)]
        sp["mu"] = float(rng.choice([0.0, 1e-5, 1e-3]))
    else:
        which = 5 if grid is not None else int(rng.choice([1, 2]))
        scale = {1: float(rng.choice([0.5, 1.0, 2.5])), 2: float(rng.choice([0.01, 0.03])), 5: float(rng.choice([0.05, 0.2, 0.8]))}[which]
        cfg = workloads.config(which, scale=scale, grid=grid)
        sp = cfg["species"][0]
        L = int(rng.choice([8, 16, 32, 64, 128, 256, 24]))
        nch = int(rng.choice([1, 2, 4])) if L % 4 == 0 and L >= 8 else 1
        cl = [L // nch] * nch
        cl[-1] += L - sum(cl)
        sp.update(n_loci=L, chrom_len=cl, r=workloads._interval_r(cl, float(rng.choice([0.01, 0.1, 0.5]))),
                  mu=float(rng.choice([0.0, 1e-3, 2e-2])))
    sp = cfg["species"][0]
    cfg["seed"] = int(rng.integers(1, 2 ** 62))
    wid = {}
    if rng.random() < 0.35:
        wid["resid_sd"] = float(rng.choice([0.1, 0.5]))
    if rng.random() < 0.35:
        wid["adult_survival"] = float(rng.choice([0.3, 0.8]))
    mating = rng.integers(0, 5)            # none / R19 / R21 (+R19) / R23 / R19 both signs
    if mating == 1:
        wid["mate_skew"] = float(rng.choice([-2.0, 1.0, 50.0]))
    elif mating == 2:
        wid["separate_sexes"] = 1
        if rng.random() < 0.5:
            wid["mate_skew"] = 1.0
    elif mating == 3:
        wid["assort"] = float(rng.choice([0.5, 4.0]))
    if rng.random() < 0.3:
        wid["mother_skew"] = float(rng.choice([-1.0, 1.5]))
    elif rng.random() < 0.25:
        wid["fec_cost"] = float(rng.choice([0.05, 0.5]))
    if rng.random() < 0.3:
        wid["monogamy"] = 1
    if rng.random() < 0.3:
        sp["gaussian"]["dtheta"] = 0.02
    sp.update(wid)
    if "separate_sexes" in wid:
        sp["fec_a"] = 2.0 * sp["fec_a"]
    sp["capacity"] = (8 if "adult_survival" in wid else 2) * sp["capacity"]
    return cfg, wid


@pytest.mark.parametrize("seed", range(60))
def test_random_configurations(oracle_mod, binding, seed):
    """Differential test on seeded random combinations of genome, patch structure and widenings:
    production kernels against the oracle, free-running, state / sexes / log / flags compared after
    2 and 7 steps; the first step also with every intermediate (debug)."""
    import numpy as np
    rng = np.random.default_rng(9000 + seed)
    cfg, wid = _random_cfg(rng)
    parity.per_step_parity(oracle_mod, binding, cfg, 1, debug=True)
    orc = oracle_mod.Oracle(cfg)
    sim = binding.Sim(cfg, debug=False)
    parity.load_initial(orc, cfg)
    parity.load_initial(sim, cfg)
    for n in (2, 5):
        orc.step(n)
        sim.step(n)
        parity.assert_logs_equal(sim.read_log(0), orc.log(0), tag=str((seed, wid)))
        parity.assert_state_equal(sim, orc, cfg, tag=str((seed, wid)))
    assert sim.status() == orc.flags
    sim.close()
