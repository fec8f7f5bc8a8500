"""CPU oracle of the Twinkle hot path -- TEST INFRASTRUCTURE ONLY (see twk_oracle.cpp's header).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this
package.  It imports nothing from paper_2501_03322_b200 and shares no code with the CUDA path.
"""
