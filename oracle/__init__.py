"""fp64 CPU oracle of the APIC closed-form reconstruction (apic_oracle), of the within-FOV reassembly
(reassemble_oracle) and of the slide-level pupil prior (pupil_prior_oracle).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It shares no code with
``paper_2407_20469_b200`` (the CUDA product path) and imports nothing from it.
"""
