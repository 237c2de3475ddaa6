"""CPU oracle: TEST INFRASTRUCTURE, not product code (see oracle/polylab_oracle.h).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import this
package.  It shares no code with paper_2604_06575_b200/csrc and never imports that package.
"""
