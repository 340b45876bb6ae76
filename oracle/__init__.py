"""Float64 CPU oracle — TEST INFRASTRUCTURE ONLY (see shifted_fresnel.py).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_1001_4309_b200 and never imports it."""
