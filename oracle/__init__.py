"""fp64 CPU oracle for the PM / NUFFT force path of DISCO-DJ II (arXiv 2510.05206).

TEST INFRASTRUCTURE ONLY.  Nothing under ``paper_2510_05206_b200/`` imports this
package; only ``tests/``, ``__graft_entry__.smoke()`` and the ``cpu_baseline`` /
``--impl reference`` legs of ``bench.py`` may.  It shares no code with the CUDA
path (no kernels, headers, tables or helpers); both sides only consume the same
seeded inputs from ``pm_inputs``.

Modules
  pm_oracle    -- scatter / gather (PAPER.md Eq. C.1, C.2, Table 1), Fourier-space
                  Poisson + gradient + deconvolution (Sec. 2.5, Table 2), interlacing,
                  full force and its reverse-mode VJP (App. C rule table).
  nufft_oracle -- brute-force non-uniform DFT force (Eq. 2.18-2.19) and the
                  exponential-of-semicircle NUFFT stage by stage (Sec. 2.5), with the
                  i k gradient or the gradient of the kernel (:264).
  dkd_oracle   -- drift-kick-drift step (Eq. 2.14) and the backward-in-time adjoint
                  step, Table 3 row by row.
  analysis_oracle -- binned (cross-)power spectrum of the interlaced, deconvolved
                  density (:375); sheet-based resampling, trilinear variant (:369-371).
"""
