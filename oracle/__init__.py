"""fp64 CPU oracle for the BiP-PRISM on-atom contraction (arxiv/paper_2607_00756).

TEST INFRASTRUCTURE -- NOT A PRODUCT PATH.  Only ``tests/``, ``__graft_entry__.smoke()``
and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` leg may import anything from this
package.  It shares no code with ``paper_2607_00756_b200/`` (the CUDA path); neither imports
the other.  The only module both use is ``bip_inputs`` (seeded synthetic problem data).

Everything here is a plain, slow, NumPy complex128 restatement of PAPER.md written to be checked
against the paper by eye, one function per equation / algorithm step, each citing its passage:

  beams.py       beam sets (eq. 5 / Alg. 4 l.1), probe coefficients (eq. 1), hex-ring parents,
                 PRISM beam subsampling, coefficient rescale and crop mask
  sibson.py      natural-neighbour weights (eq. 8) by half-plane clipping
  multislice.py  Fresnel step (eq. 2, 6), S1 build/advance, S2 build/peel (eq. 12), Alg. 1
  bip.py         windowed reconstruction (eq. 15, eq. 11), amplitudes (eq. 13-14), output modes (§2.2.6), Alg. 5
  alg3.py        Algorithm 3: beamlet-basis probe (eq. 9-10), per-scan exit multislice, cube on all G beams
  focal.py       S1 focal back-propagation to the scattering-centroid plane (reading c20), frozen-phonon mean

Readings of silent / ambiguous points follow SURVEY.md §8(c) and are listed in DESIGN.md §3.

Pins (tests/test_oracle_*.py, all ``-m "not gpu"``):
  whole forward model  : Alg. 5 with parents = all beams equals Alg. 1 brute force per scan
  S2                   : reciprocity identity eq. 12 for random w at every plane; peel == rebuild
  propagation          : Parseval for |T| = 1; vacuum closed form vs library FFT
  fresnel_propagator   : complex Gaussian-beam closed form (sign, pi, lambda, q units, l_y vs l_x) and Talbot self-imaging
                         at z_T and z_T / 2 on both axes (tests/test_oracle_propagation_pins.py)
  defocus (c4)         : the df = -50 A probe focuses 50 A below the entrance surface (one slice), df = +50 A does not
  pruned Sibson        : equals the unpruned definition on sampled rows of the configs[1] tables (1951 / 4921 parents)
  Algorithm 3          : equals Alg. 1 on every exit beam with parents = all beams; eq. 9-10 == eq. 15 + eq. 7; Parseval;
                         equals Alg. 5's cube on the detector beams when S2 is exact (tests/test_oracle_alg3.py)
  focal (c20)          : tilted window transfer function == full-grid propagation; d = 0 and the full-parent limit reproduce
                         the plain reconstruction; hand-made centroid; on-atom error halves (tests/test_oracle_focal.py)
  normalisation        : sum |psi_0|^2 = 1 ; all-G detector => I = sum |H psi|^2
  locality             : eq. 16-18 as equalities, eq. 17 as an inequality, Alg. 3 vs Alg. 2
  reducers             : sum over q_par of qEELS == map == sum over d of cube
  weights              : w >= 0, rows sum to 1, delta at parents, linear precision inside the hull, identity limit
  hex-ring             : n_radial = 4 gives 61 parents from 365 beams (tests/golden/hexring_counts.txt)
  PRISM f              : subsampled probe == exact probe replicated with period N/f (aliasing identity); crop mask
                         == per-site maps masked and summed
  MAGPHASE             : equals LINEAR for in-phase rows; exact at parents; |R|_MAGPHASE >= |R|_LINEAR
PARITY UNPINNED: the Sibson weights for beams outside the parents' convex hull (c8), the numerical value
of BiP maps at parent factor f > 1, and the focal back-propagation (the paper states neither its centroid plane nor its
padding: reading c20) have no printed value in the paper to compare against; they are pinned only as "the algorithm as
stated" plus their defining properties and the soft trends the paper reports (the error against the f = 1 map falls as
parents are added; the centroid-plane interpolation lowers the on-atom error).
"""
