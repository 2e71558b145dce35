"""FP64 CPU oracle for the MPMI-SC tick -- TEST INFRASTRUCTURE, not the product (see mpmi_oracle.h)."""
